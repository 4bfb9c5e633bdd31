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
// Three kernels: exp_window_kernel (the window sum of a segment's last t0, one tau at a time, by a
// multiplicative recurrence: the small tau), exp_moment_kernel (the same sums for groups of 16 to
// 64 neighbouring tau at once, by a Taylor expansion of the weights in 1/tau: the large tau,
// where almost all the terms are) and exp_slide_kernel (from there backwards in t0).
//
// Layout: lanes of a warp hold consecutive tau_n (same template), so the initial window is
// streamed through shared memory and broadcast exactly like exp_direct.cu; a CTA is
// (template, block of NT tau, segment of t0).  Long t0 grids with few tau (config 5) are cut
// into segments, each with its own initial sum, to fill the GPU.
#include "plan.h"

namespace tfstat {

namespace {

constexpr float kReanchor = 4.0f;  // move t_ref when (t_ref - t0_m)/tau exceeds this
constexpr float kReanchorArg = -kReanchor * 1.4426950408889634f;  // the same on (t_ref - t0_m) kexp
constexpr float kGuard = 64.0f;    // re-sum a window whose A fell below 1/kGuard of its maximum
constexpr int kSlideChunk = 128;   // atoms per bulk copy and template (4 KB); divides kPackBlock
constexpr int kSlideStages = 3;    // ring slots per CTA
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

__device__ __forceinline__ float rcp_approx_s(const float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
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

// one packed atom (32 bytes, 32-byte aligned) with ONE 256-bit load: a gather of 32 records costs
// half the L1 wavefronts of two 128-bit loads per lane
__device__ __forceinline__ void ldg_record(const ulonglong2 *p, ulonglong2 &ra, ulonglong2 &rb)
{
    asm("ld.global.nc.v4.b64 {%0,%1,%2,%3}, [%4];"
        : "=l"(ra.x), "=l"(ra.y), "=l"(rb.x), "=l"(rb.y)
        : "l"(p));
}
// the same, and a 32-bit load, pinned where they are written (volatile): the slide kernel requests
// the data of the NEXT step before it closes a cell, and the compiler must not sink the loads
// into the branch that uses them
__device__ __forceinline__ void ldg_record_now(const ulonglong2 *p, ulonglong2 &ra, ulonglong2 &rb)
{
    asm volatile("ld.global.nc.v4.b64 {%0,%1,%2,%3}, [%4];"
                 : "=l"(ra.x), "=l"(ra.y), "=l"(rb.x), "=l"(rb.y)
                 : "l"(p));
}
__device__ __forceinline__ int ldg_int_now(const int32_t *p)
{
    int v;
    asm volatile("ld.global.nc.b32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}

// ---------------------------------------------------------------------------------------
// exp_window_kernel: the window sum of the LAST t0 of every (template, segment, tau) -- more than
// 90 % of the weighted terms of the sliding form -- by a multiplicative recurrence (north_star:
// "exp/MUFU pressure is reduced by multiplicative recurrences where timestamps allow").
//
// With f_i = exp(-(t_{i+1} - t_i)/tau) the weighted sum of atoms [lo, hi) relative to its first
// atom is the backward recurrence (Horner)  S_i = x_i + f_i S_{i+1},  S_hi = 0,  S = S_lo  (f^2 for
// a2, b2, ab).  On gapless stretches f_i is ONE constant per tau, so a term costs its 7
// multiply-adds and nothing else: no exponential, no weight multiply.  f is recomputed
// (MUFU.EX2 from the integer time step) only at the atoms pack.cu has flagged: where the time
// step changes (the two edges of a gap) -- a warp-uniform branch, every lane is on the same atom.
// Every factor is <= 1 and is taken from its own time step, so nothing drifts; the rounding of a
// sum of n terms grows like sqrt(n) 2^-24 (1.5e-5 for a year of SFTs).
//
// A thread owns RT neighbouring tau values x TPC templates: one broadcast LDS.128 pair of an atom
// serves RT TPC terms.  That ratio is what the form needs: the broadcast loads return 512 bytes
// per warp instruction to the register file, and at one tau per thread the shared-memory return
// path, not the FP32 pipe, is the limit (ncu: lsu_writeback 72 %, FMA pipe 45 %: r02 profile).
// The atoms come through a ring of kSlideStages slots shared by the CTA, filled back to front by
// bulk asynchronous copies of the packed records (cp.async.bulk + mbarrier).  The sums, scaled
// to the weight exp(-(t_lo - t0)/tau) of their first atom, go to the workspace (32 bytes per
// (template, segment, tau)); exp_slide_kernel starts from them.
// ---------------------------------------------------------------------------------------
template <int NT, int RT, int TPC, bool STATS>
__device__ __forceinline__ void exp_window_body(
    const Problem &pr, const ulonglong2 *__restrict__ packed, const int n_pad,
    float4 *__restrict__ W0, const unsigned vblock, const int n_nblocks, const int n_segs,
    const int seg_len, const int n_limit, unsigned long long *__restrict__ stats)
{
    // (tau indices [0, n_limit) only: the larger ones are exp_moment_kernel's)
    constexpr int KW = kSlideChunk, NS = TPC > 2 ? 2 : kSlideStages, NW = NT / 32;
    constexpr uint32_t kTplBytes = KW * 2 * sizeof(ulonglong2);  // one template's share of a slot
    __shared__ __align__(128) ulonglong2 s_ring[NS][TPC][2 * KW];
    __shared__ __align__(8) unsigned long long s_full[NS], s_empty[NS];

    const Grid g = pr.grid;
    const Bounds &bd = pr.bounds;
    const int lane = threadIdx.x & 31;
    // vblock = (tplgrp * n_segs + seg) * n_nblocks + j, heaviest tau block (largest tau) first
    const int j = (int)(vblock % n_nblocks);
    const int seg = (int)((vblock / n_nblocks) % n_segs);
    const int tpl0 = (int)(vblock / ((int64_t)n_nblocks * n_segs)) * TPC;
    const int n_first = (n_nblocks - 1 - j) * (NT * RT);
    const int n_count = min(NT * RT, n_limit - n_first);
    const int m = min(seg * seg_len + seg_len, g.N_t0) - 1;  // the segment's last t0

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            mbar_init(smem_u32(&s_full[s]), 1);
            mbar_init(smem_u32(&s_empty[s]), NW);
        }
        mbar_fence_init();
    }
    __syncthreads();

    // templates beyond the batch (ragged last group) alias the last real one; nothing of theirs
    // is stored
    const ulonglong2 *__restrict__ rec[TPC];
#pragma unroll
    for (int q = 0; q < TPC; ++q)
        rec[q] = packed + (int64_t)min(tpl0 + q, pr.n_templates - 1) * n_pad * 2;

    // this thread's tau values: neighbours, so that their windows end within 3 (RT - 1) atoms
    const int lo_m = __ldg(bd.lo + m);
    bool n_ok[RT];
    int n[RT], hi[RT];
    float kexp[RT];
    int hi_min = 0x7fffffff, hi_max = lo_m;
#pragma unroll
    for (int r = 0; r < RT; ++r) {
        // slots beyond the grid alias the last tau of the block (nothing of theirs is stored):
        // a thread's windows then still end within a few atoms of one another
        const int slot = (int)threadIdx.x * RT + r;
        n_ok[r] = slot < n_count;
        n[r] = n_first + min(slot, n_count - 1);
        kexp[r] = (float)(-1.4426950408889634 / (double)tau_of(g, n[r]));
        hi[r] = max(hi_index(bd, g, m, n[r]), lo_m);
        hi_min = min(hi_min, hi[r]);
        hi_max = max(hi_max, hi[r]);
    }
    const int cta_e = max(hi_index(bd, g, m, n_first + n_count - 1), lo_m);  // hi is monotone in n
    const int q0 = lo_m / KW;
    const int nq = cta_e > lo_m ? (cta_e + KW - 1) / KW - q0 : 0;
    // chunks are consumed from the last (k = nq - 1) to the first: the ring is filled in that order
    auto fill = [&](const int k) {  // thread 0: chunk k -> slot (nq - 1 - k) % NS
        const int s = (nq - 1 - k) % NS;
        const uint32_t bar = smem_u32(&s_full[s]);
        mbar_expect_tx(bar, TPC * kTplBytes);
#pragma unroll
        for (int q = 0; q < TPC; ++q)
            bulk_copy(smem_u32(&s_ring[s][q][0]), rec[q] + (int64_t)(q0 + k) * KW * 2, kTplBytes, bar);
    };
    if (threadIdx.x == 0)
        for (int u = 0; u < NS && u < nq; ++u) fill(nq - 1 - u);

    // accumulators: (A, B), (Re Fa, Im Fa), (Re Fb, Im Fb), C of (tau r, template q)
    u64 s_ab[RT][TPC], s_fa[RT][TPC], s_fb[RT][TPC];
    float s_c[RT][TPC];
#pragma unroll
    for (int r = 0; r < RT; ++r)
#pragma unroll
        for (int q = 0; q < TPC; ++q) {
            s_ab[r][q] = s_fa[r][q] = s_fb[r][q] = 0ull;
            s_c[r][q] = 0.0f;
        }
    // step factor of the atom in hand, f = exp(-(t_{i+1} - t_i)/tau), and its square
    float f[RT] = {}, f2[RT] = {};
    auto step_factor = [&](const int al) {
        const int dt = __ldg(bd.t + min(al + 1, bd.n_atoms - 1)) - __ldg(bd.t + al);
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            f[r] = ex2_approx((float)dt * kexp[r]);
            f2[r] = f[r] * f[r];
        }
    };
    // one atom into the sums of tau r: S = x + f S
    auto horner = [&](const int r, const int q, const ulonglong2 ra, const ulonglong2 rb) {
        float dtc, ab;
        unpack2(ra.x, dtc, ab);
        asm("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(s_ab[r][q]) : "l"(pack2(f2[r], f2[r])), "l"(ra.y));
        asm("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(s_fa[r][q]) : "l"(pack2(f[r], f[r])), "l"(rb.x));
        asm("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(s_fb[r][q]) : "l"(pack2(f[r], f[r])), "l"(rb.y));
        s_c[r][q] = fmaf(s_c[r][q], f2[r], ab);
        // (measured: Fb, or Fa and Fb, as scalar FFMA pairs instead of FFMA2 -- fewer FMA-pipe
        // cycles, more issue slots -- is 9 % and 13 % slower)
    };
    // a bad SFT (packed as dtc = NaN on zero channels) spoils the sums of its template
    auto poison = [&](const int q, const ulonglong2 ra) {
        float dtc, ab;
        unpack2(ra.x, dtc, ab);
        if (dtc != dtc) {
#pragma unroll
            for (int r = 0; r < RT; ++r) s_c[r][q] = dtc;
        }
    };

    // ---- the few atoms at the ragged end: [hi_min, hi_r) belong to tau r only (3 per tau step) ----
    if (hi_max > hi_min) {
#pragma unroll 1
        for (int al = hi_max - 1; al >= hi_min; --al) {
            step_factor(al);
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                const ulonglong2 ra = __ldg(rec[q] + 2 * (int64_t)al), rb = __ldg(rec[q] + 2 * (int64_t)al + 1);
#pragma unroll
                for (int r = 0; r < RT; ++r)
                    if (al < hi[r]) horner(r, q, ra, rb);
                poison(q, ra);
            }
        }
    }
    if (hi_min > lo_m) step_factor(hi_min - 1);  // the factor the main loop starts with

    // ---- atoms [lo_m, hi_min), back to front, through the ring --------------------------------
#pragma unroll 1
    for (int u = 0; u < nq; ++u) {
        const int k = nq - 1 - u;  // chunk
        const int s = u % NS;
        const int cs = (q0 + k) * KW;
        // refill the slot of the chunk before this one once every warp has released it
        if (threadIdx.x == 0 && u >= 1 && u - 1 + NS < nq) {
            mbar_wait(smem_u32(&s_empty[(u - 1) % NS]), (uint32_t)((u - 1) / NS) & 1u);
            fill(nq - 1 - (u - 1 + NS));
        }
        const int x0 = max(cs, lo_m) - cs;
        const int x1 = min(cs + KW, hi_min) - cs;
        mbar_wait(smem_u32(&s_full[s]), (uint32_t)(u / NS) & 1u);
#pragma unroll 4
        for (int i = x1 - 1; i >= x0; --i) {
            ulonglong2 ra[TPC], rb[TPC];
            unsigned flag = 0u;
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                ra[q] = s_ring[s][q][2 * i];
                rb[q] = s_ring[s][q][2 * i + 1];
                flag |= (unsigned)(ra[q].x & 0x80000000ull);
            }
            if (flag) {  // warp-uniform, rare: the time step changes here, or a bad SFT
                step_factor(cs + i);
#pragma unroll
                for (int q = 0; q < TPC; ++q) poison(q, ra[q]);
            }
#pragma unroll
            for (int r = 0; r < RT; ++r)
#pragma unroll
                for (int q = 0; q < TPC; ++q) horner(r, q, ra[q], rb[q]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&s_empty[s]));
    }

    // ---- scale to the weight of the first atom and store ---------------------------------------
    const int t_ref = (int)t0_of(g, m);
    const int t_lo = __ldg(bd.t + min(lo_m, bd.n_atoms - 1));
#pragma unroll
    for (int r = 0; r < RT; ++r) {
        if (!n_ok[r]) continue;
        const float e0 = hi[r] > lo_m ? ex2_approx((float)(t_lo - t_ref) * kexp[r]) : 0.0f;
        const float e02 = e0 * e0;
#pragma unroll
        for (int q = 0; q < TPC; ++q) {
            if (tpl0 + q >= pr.n_templates) continue;
            float A, B, far, fai, fbr, fbi;
            unpack2(s_ab[r][q], A, B);
            unpack2(s_fa[r][q], far, fai);
            unpack2(s_fb[r][q], fbr, fbi);
            float4 *__restrict__ dst =
                W0 + (((int64_t)(tpl0 + q) * n_segs + seg) * g.N_tau + n[r]) * 2;
            dst[0] = make_float4(A * e02, B * e02, s_c[r][q] * e02, far * e0);
            dst[1] = make_float4(fai * e0, fbr * e0, fbi * e0, 0.0f);
        }
    }
    if (STATS) {
        unsigned long long nt = 0;
#pragma unroll
        for (int r = 0; r < RT; ++r) nt += n_ok[r] ? (unsigned long long)(hi[r] - lo_m) : 0ull;
        nt *= (unsigned long long)min(TPC, pr.n_templates - tpl0);
#pragma unroll
        for (int sft = 16; sft >= 1; sft >>= 1) nt += __shfl_xor_sync(0xffffffffu, nt, sft);
        if (lane == 0 && nt) atomicAdd(stats + 0, nt);
    }
}

// ---------------------------------------------------------------------------------------
// exp_moment_kernel: the same window sums for GROUPS of R neighbouring tau values at once, by a
// Taylor expansion of the weights in 1/tau about the group's centre.
//
// With u = 1/tau, u_c the centre of the group's u range, d_max its half width and s = t - t_lo,
//     exp(-s u_n) = exp(-s u_c) exp(-s (u_n - u_c)) = e(s) sum_k (-rho_n)^k z(s)^k / k!,
//     z = s d_max  (>= 0),   rho_n = (u_n - u_c) / d_max  in [-1, 1],
// so the window sums of ALL tau_n of the group are combinations of 8 moments that do not depend
// on n:  Q_k = sum_a e_a z_a^k / k! x_a  (e^2 and (2z)^k for a2, b2, ab),
//     S_n = sum_{k<8} (-rho_n)^k Q_k  + the few atoms of [hi_{n0}, hi_n) (added to the moments as n
// grows).  A window is at most 3 tau long, so z <= 1.5 (R - 1) dtau / tau; the plan (api.cu)
// takes a group size R in {16, 32, 64} only where that is <= 0.17: the truncation error of
// a WEIGHT is then below (2 x 0.17)^8 / 8! = 4.4e-9 relative (the squared weights are the worse
// case), a tenth of the fp32 rounding of the sums it enters (DESIGN.md 6.2 has the numbers).
// Every weight is positive and evaluated from its own time stamp with one MUFU.EX2: nothing
// drifts, gaps are just time stamps.  Work per atom and template: 8 x 7 multiply-adds for R tau
// values instead of 7 R.
//
// A thread owns HALF the moments of one group -- the even powers (lane & 1 = 0) or the odd ones
// -- for TPC = 2 templates: 4 x 7 x 2 accumulators, so that one broadcast LDS.128 pair of an
// atom serves 56 multiply-adds as in exp_window_kernel.  A warp is 8 groups x 2 halves x 2
// template pairs (a half-warp per pair, so every quarter-warp phase of an LDS.128 still reads one
// address).  That is few threads (config 4: 46 per template pair), each with a long loop, so
// the 4 warps of a CTA share the SAME groups and templates and split the atoms between them,
// chunk k to warp k mod 4, each through its own ring of bulk asynchronous copies (as the split
// form of exp_direct.cu): moments are plain sums, so the partial ones meet in shared memory.
// Then every warp finishes a quarter of the group's tau values.
// ---------------------------------------------------------------------------------------
constexpr int kMomKW = 32;   // atoms per bulk copy and template (1 KB); divides kPackBlock
constexpr int kMomGW = 8;    // groups per warp
constexpr int kMomNS = 2;    // ring slots per warp
constexpr int kMomNW = 4;    // warps per CTA: they split the atoms of the same windows
static_assert(kPackBlock % kMomKW == 0, "a staged chunk must lie inside one packed time block");

struct MomAcc {  // one moment of one template
    u64 ab, fa, fb;
    float c;
};

// tau indices [n16, n32) in groups of 16, [n32, n64) in groups of 32, [n64, N_tau) in groups of 64
template <bool STATS>
__global__ void __launch_bounds__(32 * kMomNW, 4)
    exp_moment_kernel(const __grid_constant__ Problem pr, const ulonglong2 *__restrict__ packed,
                      const int n_pad, float4 *__restrict__ W0, const int n16, const int n32,
                      const int n64,
                      const int n_gblocks, const int n_segs, const int seg_len,
                      unsigned long long *__restrict__ stats)
{
    constexpr int TPC = 2, KW = kMomKW, NS = kMomNS;
    constexpr uint32_t kTplBytes = KW * 2 * sizeof(ulonglong2);
    // a warp's ring slot: [pair][template of the pair][records]
    __shared__ __align__(128) ulonglong2 s_ring[kMomNW][NS][2][TPC][2 * KW];
    __shared__ __align__(8) unsigned long long s_bar[kMomNW][NS];

    const Grid &g = pr.grid;
    const Bounds &bd = pr.bounds;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int h = lane & 1;    // 0: powers 0, 2, 4, 6;  1: powers 1, 3, 5, 7
    const int tp = lane >> 4;  // which of the warp's two template pairs
    // blockIdx = (tplquad * n_segs + seg) * n_gblocks + gb, heaviest groups (largest tau) first
    const int gb = (int)(blockIdx.x % n_gblocks);
    const int seg = (int)((blockIdx.x / n_gblocks) % n_segs);
    const int quad0 = (int)(blockIdx.x / ((int64_t)n_gblocks * n_segs)) * 2 * TPC;
    // a pair beyond the batch aliases the last one (nothing of its is stored)
    const int tpl0 = quad0 + tp * TPC;
    const bool tp_ok = tpl0 < pr.n_templates;
    // groups, from the largest tau down: G64 of 64 tau values, then G32 of 32, then G16 of 16
    const int G64 = (g.N_tau - n64 + 63) / 64, G32 = (n64 - n32 + 31) / 32, G16 = (n32 - n16 + 15) / 16;
    const int gx = gb * kMomGW + ((lane >> 1) & (kMomGW - 1));
    const bool g_ok = gx < G64 + G32 + G16;
    const int gi = g_ok ? gx : G64 + G32 + G16 - 1;  // no group: alias the lightest one
    const int R = gi < G64 ? 64 : gi < G64 + G32 ? 32 : 16;
    const int n0 = gi < G64         ? n64 + (G64 - 1 - gi) * 64
                   : gi < G64 + G32 ? n32 + (G64 + G32 - 1 - gi) * 32
                                    : n16 + (G64 + G32 + G16 - 1 - gi) * 16;
    const int Rg = min(R, (gi < G64 ? g.N_tau : gi < G64 + G32 ? n64 : n32) - n0);
    const int m = min(seg * seg_len + seg_len, g.N_t0) - 1;  // the segment's last t0

    const uint32_t bar0 = smem_u32(&s_bar[warp][0]);
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(bar0 + 8 * s, 1);
        mbar_fence_init();
    }
    __syncwarp();

    const ulonglong2 *__restrict__ rec[TPC];
#pragma unroll
    for (int q = 0; q < TPC; ++q)
        rec[q] = packed + (int64_t)min(tpl0 + q, pr.n_templates - 1) * n_pad * 2;
    // (lane 0 fills the ring for BOTH pairs of the warp)
    const ulonglong2 *__restrict__ rec_fill[2][TPC];
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int q = 0; q < TPC; ++q)
            rec_fill[a][q] =
                packed + (int64_t)min(quad0 + a * TPC + q, pr.n_templates - 1) * n_pad * 2;

    // the group's expansion: u_c, d_max from its first and last tau (double, then fp32)
    const double u_first = 1.0 / (double)tau_of(g, n0), u_last = 1.0 / (double)tau_of(g, n0 + Rg - 1);
    const double u_c = 0.5 * (u_first + u_last), d_max = 0.5 * (u_first - u_last);
    const float kc = (float)(-1.4426950408889634 * u_c);  // e = 2^(s kc)
    const float dm = (float)d_max;                        // z = s dm
    // steps between this thread's powers k, k + 2, k + 4, k + 6:  z^2 / ((k + 1)(k + 2))
    const float c1 = h ? 1.0f / 6.0f : 0.5f, c2 = h ? 0.05f : 1.0f / 12.0f,
                c3 = h ? 1.0f / 42.0f : 1.0f / 30.0f;

    const int lo_m = __ldg(bd.lo + m);
    const int t_lo = __ldg(bd.t + min(lo_m, bd.n_atoms - 1));
    const int hi1 = max(hi_index(bd, g, m, n0), lo_m);  // end of the group's SHORTEST window

    MomAcc acc[4][TPC];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int q = 0; q < TPC; ++q) {
            acc[j][q].ab = acc[j][q].fa = acc[j][q].fb = 0ull;
            acc[j][q].c = 0.0f;
        }
    // one atom into the thread's four moments of both templates; dt = t - t_lo (finite), e its
    // weight (0 for an atom outside this thread's window)
    auto add_atom = [&](const float e, const float z, const ulonglong2 (&ra)[TPC],
                        const ulonglong2 (&rb)[TPC]) {
        const float zz = z * z;
        float p[4], s2[4];
        p[0] = e * (h ? z : 1.0f);
        s2[0] = p[0] * (e * (h ? 2.0f : 1.0f));  // e^2 (2z)^k / k!
        const float zc1 = zz * c1, zc2 = zz * c2, zc3 = zz * c3;
        p[1] = p[0] * zc1;
        p[2] = p[1] * zc2;
        p[3] = p[2] * zc3;
        s2[1] = s2[0] * (4.0f * zc1);
        s2[2] = s2[1] * (4.0f * zc2);
        s2[3] = s2[2] * (4.0f * zc3);
#pragma unroll
        for (int q = 0; q < TPC; ++q) {
            float dtc, ab;
            unpack2(ra[q].x, dtc, ab);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                ffma2(acc[j][q].ab, pack2(s2[j], s2[j]), ra[q].y);
                ffma2(acc[j][q].fa, pack2(p[j], p[j]), rb[q].x);
                ffma2(acc[j][q].fb, pack2(p[j], p[j]), rb[q].y);
                acc[j][q].c = fmaf(s2[j], ab, acc[j][q].c);
            }
        }
    };
    // a bad SFT (packed as dtc = NaN on zero channels) spoils the sums of its template
    auto poison = [&](const int q) { acc[0][q].c = nanf(""); };

    // ---- phase 1: atoms [lo_m, hi1), chunk k by warp k mod kMomNW through its ring -------------
    const int warp_e = __reduce_max_sync(0xffffffffu, hi1);
    const int q0 = lo_m / KW;
    const int nq = warp_e > lo_m ? (warp_e + KW - 1) / KW - q0 : 0;
    auto fill = [&](const int k) {  // lane 0: chunk k -> slot (k / kMomNW) % NS
        const int s = (k / kMomNW) % NS;
        mbar_expect_tx(bar0 + 8 * s, 2 * TPC * kTplBytes);
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int q = 0; q < TPC; ++q)
                bulk_copy(smem_u32(&s_ring[warp][s][a][q][0]),
                          rec_fill[a][q] + (int64_t)(q0 + k) * KW * 2, kTplBytes, bar0 + 8 * s);
    };
    if (lane == 0)
        for (int u = 0; u < NS && warp + u * kMomNW < nq; ++u) fill(warp + u * kMomNW);
#pragma unroll 1
    for (int k = warp, u = 0; k < nq; k += kMomNW, ++u) {
        const int s = u % NS;
        const int cs = (q0 + k) * KW;  // first atom of the chunk
        // s = t - t_lo = dtc + (t_block - t_lo): one FMA each for the exponent and for z
        const int tb = __ldg(bd.t + cs - cs % kPackBlock);
        const float sb = (float)(tb - t_lo);
        const float cc = sb * kc, cz = sb * dm;
        const int x0 = max(cs, lo_m) - cs;
        const int x1 = min(cs + KW, warp_e) - cs;
        mbar_wait(bar0 + 8 * s, (uint32_t)(u / NS) & 1u);
#pragma unroll 2
        for (int i = x0; i < x1; ++i) {
            ulonglong2 ra[TPC], rb[TPC];
            unsigned flag = 0u;
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                ra[q] = s_ring[warp][s][tp][q][2 * i];
                rb[q] = s_ring[warp][s][tp][q][2 * i + 1];
                flag |= (unsigned)(ra[q].x & 0x80000000ull);
            }
            flag = __any_sync(0xffffffffu, flag != 0u);  // (the two pairs may differ: bad SFTs)
            const bool inside = cs + i < hi1;
            float dtc = fabsf(__uint_as_float((unsigned)ra[0].x));
            if (flag) {  // warp-uniform, rare: a gap edge (nothing to do) or a bad SFT
                bool any_bad = false;
#pragma unroll
                for (int q = 0; q < TPC; ++q) {
                    const float d = __uint_as_float((unsigned)ra[q].x);
                    if (d != d) {
                        any_bad = true;
                        if (inside) poison(q);
                    }
                }
                if (any_bad) dtc = (float)(__ldg(bd.t + cs + i) - tb);  // the record's is NaN
            }
            const float e = inside ? ex2_approx(fmaf(dtc, kc, cc)) : 0.0f;
            add_atom(e, fmaf(dtc, dm, cz), ra, rb);
        }
        __syncwarp();  // every lane is done with the slot: refill it
        if (lane == 0 && k + NS * kMomNW < nq) fill(k + NS * kMomNW);
    }

    // ---- the warps' partial moments meet in shared memory (the rings are done with); every warp
    // leaves with the full sums
    {
        float *red = reinterpret_cast<float *>(&s_ring[0][0][0][0][0]);  // [NW][56][32]
        static_assert(sizeof(s_ring) >= sizeof(float) * kMomNW * 56 * 32, "reduction buffer");
        __syncthreads();
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                float v[7];
                unpack2(acc[j][q].ab, v[0], v[1]);
                unpack2(acc[j][q].fa, v[2], v[3]);
                unpack2(acc[j][q].fb, v[4], v[5]);
                v[6] = acc[j][q].c;
#pragma unroll
                for (int c = 0; c < 7; ++c) red[(warp * 56 + (j * TPC + q) * 7 + c) * 32 + lane] = v[c];
            }
        __syncthreads();
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                float v[7];
#pragma unroll
                for (int c = 0; c < 7; ++c) {
                    float t = 0.0f;
#pragma unroll
                    for (int w = 0; w < kMomNW; ++w) t += red[(w * 56 + (j * TPC + q) * 7 + c) * 32 + lane];
                    v[c] = t;
                }
                acc[j][q].ab = pack2(v[0], v[1]);
                acc[j][q].fa = pack2(v[2], v[3]);
                acc[j][q].fb = pack2(v[4], v[5]);
                acc[j][q].c = v[6];
            }
    }

    // ---- phase 2: tau by tau -- the atoms [hi_{n-1}, hi_n) join the moments (a gather per lane:
    // every group is at its own place by now), then S_n = sum_k (-rho_n)^k Q_k ------------------
    // (warp w takes the tau values [w R/4, (w + 1) R/4) of every group: it first catches up with
    // the atoms of the tau values before its own)
    const int t_ref = (int)t0_of(g, m);
    int hi_prev = hi1;
    // (a group of 64 takes 16 steps per warp, one of 32 eight, one of 16 four: the lanes of the
    // shorter ones idle through the rest, the shuffles below need every lane)
    const int RQ = R / kMomNW;
    const int steps = __reduce_max_sync(0xffffffffu, RQ);
#pragma unroll 1
    for (int it = warp ? -1 : 0; it < steps; ++it) {
        const bool catch_up = it < 0;  // only extends the moments, stores nothing
        const bool mine = it < RQ;
        const int qn = warp * RQ + min(it, RQ - 1);
        // (lanes beyond their group's last tau repeat it)
        const int n = n0 + min(qn, Rg - 1);
        const int hi_n = max(hi_index(bd, g, m, n), lo_m);
        for (int al = hi_prev; al < hi_n; ++al) {
            ulonglong2 ra[TPC], rb[TPC];
#pragma unroll
            for (int q = 0; q < TPC; ++q) ldg_record(rec[q] + 2 * (int64_t)al, ra[q], rb[q]);
            const float sdt = (float)(__ldg(bd.t + al) - t_lo);
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                const float d = __uint_as_float((unsigned)ra[q].x);
                if (d != d) poison(q);
            }
            add_atom(ex2_approx(sdt * kc), sdt * dm, ra, rb);
        }
        hi_prev = max(hi_prev, hi_n);
        if (catch_up) continue;  // (warp-uniform)
        // this thread's powers of -rho: (-rho)^h, then steps of rho^2
        const double un = 1.0 / (double)tau_of(g, n);
        const float rho = d_max > 0.0 ? (float)((un - u_c) / d_max) : 0.0f;
        const float r2 = rho * rho;
        float cj[4];
        cj[0] = h ? -rho : 1.0f;
        cj[1] = cj[0] * r2;
        cj[2] = cj[1] * r2;
        cj[3] = cj[2] * r2;
        float S[TPC][7];
#pragma unroll
        for (int q = 0; q < TPC; ++q) {
#pragma unroll
            for (int c = 0; c < 7; ++c) S[q][c] = 0.0f;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float A, B, far, fai, fbr, fbi;
                unpack2(acc[j][q].ab, A, B);
                unpack2(acc[j][q].fa, far, fai);
                unpack2(acc[j][q].fb, fbr, fbi);
                S[q][0] = fmaf(cj[j], A, S[q][0]);
                S[q][1] = fmaf(cj[j], B, S[q][1]);
                S[q][2] = fmaf(cj[j], acc[j][q].c, S[q][2]);
                S[q][3] = fmaf(cj[j], far, S[q][3]);
                S[q][4] = fmaf(cj[j], fai, S[q][4]);
                S[q][5] = fmaf(cj[j], fbr, S[q][5]);
                S[q][6] = fmaf(cj[j], fbi, S[q][6]);
            }
#pragma unroll
            for (int c = 0; c < 7; ++c) S[q][c] += __shfl_xor_sync(0xffffffffu, S[q][c], 1);
        }
        // scaled to the weight exp(-(t_lo - t0)/tau_n) of the window's first atom, as
        // exp_window_kernel stores them; the even lane stores template 0, the odd one template 1
        if (g_ok && mine && qn < Rg && tp_ok && tpl0 + h < pr.n_templates) {
            const float kexp = (float)(-1.4426950408889634 * un);
            const float e0 = hi_n > lo_m ? ex2_approx((float)(t_lo - t_ref) * kexp) : 0.0f;
            const float e02 = e0 * e0;
            float Sq[7];
#pragma unroll
            for (int c = 0; c < 7; ++c) Sq[c] = h ? S[1][c] : S[0][c];
            float4 *__restrict__ dst = W0 + (((int64_t)(tpl0 + h) * n_segs + seg) * g.N_tau + n) * 2;
            dst[0] = make_float4(Sq[0] * e02, Sq[1] * e02, Sq[2] * e02, Sq[3] * e0);
            dst[1] = make_float4(Sq[4] * e0, Sq[5] * e0, Sq[6] * e0, 0.0f);
        }
    }
    if (STATS) {
        // moment terms: (atom, power, template) triples of 7 multiply-adds each
        const int hi_last = max(hi_index(bd, g, m, n0 + Rg - 1), lo_m);
        unsigned long long nt = (g_ok && tp_ok && warp == 0)
                                    ? (unsigned long long)(hi_last - lo_m) * 4ull *
                                          (unsigned long long)min(TPC, pr.n_templates - tpl0)
                                    : 0ull;
#pragma unroll
        for (int sft = 16; sft >= 1; sft >>= 1) nt += __shfl_xor_sync(0xffffffffu, nt, sft);
        if (lane == 0 && nt) atomicAdd(stats + TFSTAT_STAT_MOMENT, nt);
    }
}

// ---------------------------------------------------------------------------------------
// exp_slide_kernel: a thread owns one tau x TPC templates, starts from the window sums of the
// segment's last t0 (exp_window_kernel) and slides backwards in t0.  The weights E_a depend on
// (atom, tau) only, so one MUFU.EX2 (+ its argument and E^2) serves the TPC templates.
//
// A t0 step is a chain of dependent loads (row start -> window end -> atom records) in front of
// the arithmetic, so the indices of the step m -> m - 1 are requested one step ahead and the
// record of the leaving atom BEFORE cell m is closed.
//
// FAST PATH, taken when every lane of the warp is in the common case -- at most one atom enters
// and one leaves, the windows of m and m - 1 overlap, t_ref stays, every cell of the warp is
// well conditioned: straight-line code.  The entering atom is the same for all lanes (it depends
// on t0 only): each warp stages 32 of them at a time in shared memory (coalesced, once per 32
// steps) and reads them back by broadcast; the leaving atom is one gather per lane, one 256-bit
// load per template.  An atom that does not exist (n_in = 0, n_out = 0) is read from a clamped
// address and gets the weight 0 by a select.  Cells are closed in fp32 and the lanes VOTE on
// whether any of them needs the careful closure; the marginals are updated without branches.
// Everything else (several atoms per step, disjoint windows, re-anchoring, ill-conditioned or
// short cells, the segment's first row, re-summing a window that lost its weight) is in two
// functions that are NOT inlined and work on a copy of the thread's state in local memory, so
// that the register allocation of the loop is that of the fast path alone.  ncu on config 4
// with everything in one loop body: 304 warp instructions per step, of which 50
// BRA/BSSY/BSYNC, 47 integer compares and 21 spill loads/stores; L1 wavefronts 62 % of peak.
// ---------------------------------------------------------------------------------------
constexpr float kHalfLog2eS = 0.72134752044448170368f;  // log2(e) / 2: F log2e = 2F * this

template <int TPC>
struct SlideState {
    SlideAcc acc[TPC];
    float A_max[TPC];
    // marginals per template: running max (ties: a thread's rows only decrease, so the later cell
    // wins), the row of the best cell, log-sum-exp against a reference that moves rarely, and the
    // number of cells that do not count (flagged ones)
    float mg_best[TPC], mg_ref2[TPC], mg_sum[TPC];
    int32_t mg_m[TPC], n_bad[TPC];
    int m, lo_m, hi, lo2, hi2, t_ref;
    unsigned n_term[4];  // STATS: (window), enter, leave, re-sum (x TPC templates)
};

struct SlideCtx {  // what a thread's cold paths need besides its state
    const ulonglong2 *packed;
    int n_pad, tpl0, n, n_ok, m_beg;
    float kexp;
};

template <int TPC>
__device__ __forceinline__ void slide_copy(SlideState<TPC> &d, const SlideState<TPC> &s)
{
#pragma unroll
    for (int q = 0; q < TPC; ++q) {
        d.acc[q].ab = s.acc[q].ab;
        d.acc[q].fa = s.acc[q].fa;
        d.acc[q].fb = s.acc[q].fb;
        d.acc[q].c = s.acc[q].c;
        d.A_max[q] = s.A_max[q];
        d.mg_best[q] = s.mg_best[q];
        d.mg_ref2[q] = s.mg_ref2[q];
        d.mg_sum[q] = s.mg_sum[q];
        d.mg_m[q] = s.mg_m[q];
        d.n_bad[q] = s.n_bad[q];
    }
    d.m = s.m;
    d.lo_m = s.lo_m;
    d.hi = s.hi;
    d.lo2 = s.lo2;
    d.hi2 = s.hi2;
    d.t_ref = s.t_ref;
#pragma unroll
    for (int i = 0; i < 4; ++i) d.n_term[i] = s.n_term[i];
}

// acc += sign * E x for one atom read straight from the packed records, one weight for the TPC
// templates
template <int TPC>
__device__ __forceinline__ void slide_add_global(SlideState<TPC> &s, const Bounds &bd,
                                                 const ulonglong2 *const (&rec)[TPC],
                                                 const float kexp, const int al, const float sign)
{
    const float e = ex2_approx((float)(__ldg(bd.t + al) - s.t_ref) * kexp);
#pragma unroll
    for (int q = 0; q < TPC; ++q) {
        const ulonglong2 ra = __ldg(rec[q] + 2 * (int64_t)al), rb = __ldg(rec[q] + 2 * (int64_t)al + 1);
        float dtc, ab;
        unpack2(ra.x, dtc, ab);
        const float eq = fmaf(dtc, 0.0f, e);  // NaN for an atom that is not finite (pack.cu)
        const float w = sign * eq;
        acc_add(s.acc[q], w, w * eq, ra, rb);
    }
}

// a window summed afresh (t_ref = the t0 of row m - 1): lanes whose window lost most of its
// weight, or does not overlap its neighbour
template <int TPC, bool STATS>
__device__ __noinline__ void slide_resum(SlideState<TPC> &s, const Problem &pr, const SlideCtx &c)
{
    const ulonglong2 *rec[TPC];
#pragma unroll
    for (int q = 0; q < TPC; ++q) {
        rec[q] = c.packed + (int64_t)min(c.tpl0 + q, pr.n_templates - 1) * c.n_pad * 2;
        acc_zero(s.acc[q]);
    }
    s.t_ref = (int)t0_of(pr.grid, s.m - 1);
    for (int al = s.lo2; al < s.hi2; ++al) slide_add_global<TPC>(s, pr.bounds, rec, c.kexp, al, 1.0f);
    if (STATS) s.n_term[3] += (unsigned)(s.hi2 - s.lo2);
#pragma unroll
    for (int q = 0; q < TPC; ++q) {
        float A, B;
        unpack2(s.acc[q].ab, A, B);
        s.A_max[q] = A;
    }
}

// one t0 step the careful way: closure of cell (m, n) with closure_2F_exp where fp32 does not
// do, then the sums move on to row m - 1 with loops over the entering and leaving atoms.
// Returns true after the segment's first row.
template <int TPC, bool STATS>
__device__ __noinline__ bool slide_step_generic(SlideState<TPC> &s, const Problem &pr,
                                                const SlideCtx &c)
{
    const Grid &g = pr.grid;
    const Bounds &bd = pr.bounds;
    const int m = s.m, n = c.n;
    const ulonglong2 *rec[TPC];
#pragma unroll
    for (int q = 0; q < TPC; ++q)
        rec[q] = c.packed + (int64_t)min(c.tpl0 + q, pr.n_templates - 1) * c.n_pad * 2;
    const int64_t cells = (int64_t)g.N_t0 * g.N_tau;
    const int32_t flat = m * g.N_tau + n;
    const int cnt = s.hi - s.lo_m;

    // ---- a4 + a5 of cell (m, n) of every template
#pragma unroll
    for (int q = 0; q < TPC; ++q) {
        float A, B, far, fai, fbr, fbi;
        unpack2(s.acc[q].ab, A, B);
        unpack2(s.acc[q].fa, far, fai);
        unpack2(s.acc[q].fb, fbr, fbi);
        const float C = s.acc[q].c;
        // the fast path's arithmetic, so that a cell's value does not depend on its neighbours
        const float p = A * B;
        const float D = fmaf(-C, C, p);
        const float na = fmaf(far, far, fai * fai);
        const float nb = fmaf(fbr, fbr, fbi * fbi);
        const float re = fmaf(far, fbr, fai * fbi);
        float num = B * na;
        num = fmaf(A, nb, num);
        num = fmaf(-2.0f * C, re, num);
        float twoF = 2.0f * num * rcp_approx_s(D);
        uint32_t fl = 0u;
        if (!(D > 0.015625f * p && p > 1.0e-30f && p < 1.0e30f && cnt >= pr.min_atoms &&
              fabsf(twoF) < 3.0e38f)) {
            const int tq = min(c.tpl0 + q, pr.n_templates - 1);
            twoF = closure_2F_exp<false>(A, B, C, far, fai, fbr, fbi, s.lo_m, cnt, pr.min_atoms, fl,
                                         pr.atoms + (int64_t)tq * pr.template_stride, pr.ld, bd.t,
                                         t0_of(g, m), (double)tau_of(g, n));
        }
        if (c.n_ok && c.tpl0 + q < pr.n_templates) {
            const int64_t o = (int64_t)(c.tpl0 + q) * cells + flat;
            if (pr.out_maps) pr.out_maps[o] = twoF;
            if (pr.out_flags) pr.out_flags[o] = (uint8_t)fl;
        }
        if (!fl) {
            if (twoF >= s.mg_best[q]) {
                s.mg_best[q] = twoF;
                s.mg_m[q] = m;
            }
            if (fmaf(twoF, kHalfLog2eS, -s.mg_ref2[q]) > 60.0f) {  // move the reference
                s.mg_sum[q] *= ex2_approx(s.mg_ref2[q] - twoF * kHalfLog2eS);
                s.mg_ref2[q] = twoF * kHalfLog2eS;
            }
            s.mg_sum[q] += ex2_approx(fmaf(twoF, kHalfLog2eS, -s.mg_ref2[q]));
        } else {
            s.n_bad[q] += 1;
        }
    }
    if (m == c.m_beg) return true;

    // ---- the sums move on to cell m - 1
    int lo3 = s.lo2, hi3 = s.hi2;
    if (m - 1 > c.m_beg) {
        lo3 = __ldg(bd.lo + m - 2);
        hi3 = max(hi_index(bd, g, m - 2, n), lo3);
    }
    const int lo2 = s.lo2, hi2 = s.hi2, lv = max(hi2, s.lo_m);
    bool fresh = (hi2 <= s.lo_m) || (hi2 == lo2);  // no overlap with window m, or empty
    if (!fresh) {
        const int t0_2 = (int)t0_of(g, m - 1);
        const float sh = (float)(s.t_ref - t0_2);
        if (sh * c.kexp < kReanchorArg) {  // keep the weights of entering atoms <= e^kReanchor
            const float sc = ex2_approx(sh * c.kexp);
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                acc_scale(s.acc[q], sc);
                s.A_max[q] *= sc * sc;
            }
            s.t_ref = t0_2;
        }
        for (int al = lo2; al < s.lo_m; ++al)  // entering, low end
            slide_add_global<TPC>(s, bd, rec, c.kexp, al, 1.0f);
        for (int al = lv; al < s.hi; ++al)  // leaving, high end
            slide_add_global<TPC>(s, bd, rec, c.kexp, al, -1.0f);
        if (STATS) {
            s.n_term[1] += (unsigned)(s.lo_m - lo2);
            s.n_term[2] += (unsigned)max(s.hi - lv, 0);
        }
#pragma unroll
        for (int q = 0; q < TPC; ++q) {
            float A, B;
            unpack2(s.acc[q].ab, A, B);
            s.A_max[q] = fmaxf(s.A_max[q], A);
            // a window that lost most of its weight is re-summed (for all TPC templates: a fresh
            // sum is always right); written so that a NaN / inf atom in the running sums also
            // forces a fresh sum: once it has left the window it must not linger
            fresh = fresh || !(A * kGuard >= s.A_max[q]);
        }
    }
    if (fresh) slide_resum<TPC, STATS>(s, pr, c);
    s.m = m - 1;
    s.lo_m = lo2;
    s.hi = hi2;
    s.lo2 = lo3;
    s.hi2 = hi3;
    return false;
}

template <int NT, int TPC, bool STATS>
__device__ __forceinline__ void exp_slide_body(
    const Problem &pr, const ulonglong2 *__restrict__ packed, const int n_pad,
    const float4 *W0, Partial *__restrict__ partials, const unsigned vblock, const int n_nblocks,
    const int n_segs, const int seg_len, unsigned long long *__restrict__ stats)
{
    constexpr unsigned kFull = 0xffffffffu;
    constexpr int NW = NT / 32;
    __shared__ Marg s_red[32];
    __shared__ __align__(16) ulonglong2 s_in[NW][TPC][64];  // a warp's next 32 entering atoms
    __shared__ int s_tin[NW][32];                           // and their time stamps

    const Grid &g = pr.grid;
    const Bounds &bd = pr.bounds;
    const int lane = threadIdx.x & 31;
    const int warp = (int)threadIdx.x >> 5;
    // vblock = (tplgrp * n_segs + seg) * n_nblocks + j, heaviest tau block (largest tau) first
    const int j = (int)(vblock % n_nblocks);
    const int seg = (int)((vblock / n_nblocks) % n_segs);
    const int tpl0 = (int)(vblock / ((int64_t)n_nblocks * n_segs)) * TPC;
    const int n_first = (n_nblocks - 1 - j) * NT;
    const int n_count = min(NT, g.N_tau - n_first);
    const int m_beg = seg * seg_len;
    const int m_end = min(m_beg + seg_len, g.N_t0);

    // Templates beyond the batch (ragged last group) alias the last real one, tau slots beyond
    // the grid alias the block's last tau: they run the same instructions as their neighbours
    // (the fast path is taken warp by warp) and nothing of theirs is stored.
    const ulonglong2 *__restrict__ rec[TPC];
#pragma unroll
    for (int q = 0; q < TPC; ++q)
        rec[q] = packed + (int64_t)min(tpl0 + q, pr.n_templates - 1) * n_pad * 2;
    const bool n_ok = (int)threadIdx.x < n_count;
    const int n = n_first + min((int)threadIdx.x, n_count - 1);
    const float kexp = (float)(-1.4426950408889634 / (double)tau_of(g, n));
    const int a_last = bd.n_atoms - 1;
    // window end of cell (mm, n): one entry of the lattice table (bounds.cu), else a binary search
    const bool has_edge = bd.edge != nullptr;
    const int jn = n * bd.e_n;  // (the lattice has at most 2^22 points: 32-bit indices)
    int in_base = 0x40000000;   // first atom of the warp's staged entering atoms (none yet)

    // ---- the segment's last cell (m_end - 1, n): its window sums come from exp_window_kernel ----
    SlideState<TPC> s;
    s.m = m_end - 1;
    s.lo_m = __ldg(bd.lo + s.m);
    s.hi = max(hi_index(bd, g, s.m, n), s.lo_m);
    s.t_ref = (int)t0_of(g, s.m);  // seconds (int32: every grid time fits, TFSTAT_EOVERFLOW otherwise)
#pragma unroll
    for (int q = 0; q < TPC; ++q) {
        const int tq = min(tpl0 + q, pr.n_templates - 1);
        const float4 *w = W0 + (((int64_t)tq * n_segs + seg) * g.N_tau + n) * 2;
        const float4 w0 = w[0], w1 = w[1];
        s.acc[q].ab = pack2(w0.x, w0.y);
        s.acc[q].c = w0.z;
        s.acc[q].fa = pack2(w0.w, w1.x);
        s.acc[q].fb = pack2(w1.y, w1.z);
        s.A_max[q] = w0.x;
        s.mg_best[q] = -INFINITY;
        s.mg_m[q] = 0;
        s.mg_ref2[q] = -1.0e30f;
        s.mg_sum[q] = 0.0f;
        s.n_bad[q] = 0;
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) s.n_term[i] = 0u;
    s.lo2 = s.lo_m;
    s.hi2 = s.hi;
    if (s.m > m_beg) {
        s.lo2 = __ldg(bd.lo + s.m - 1);
        s.hi2 = max(hi_index(bd, g, s.m - 1, n), s.lo2);
    }

    // ---- slide backwards in t0: closure of cell m, then step to m - 1 ------------------------
    // (a warp whose tau slots all lie beyond the grid has nothing to do but the final reduction)
    // The fast path is a tight loop of its own, left through one of two cold exits.  (ptxas still
    // ends every step with ~45 register moves -- it builds the new sums next to the old ones and
    // copies them back -- which neither this loop shape nor forcing eq. (7) in front of the
    // update changes.)
    bool finished = !(warp * 32 < n_count);
#pragma unroll 1
    while (!finished) {
        int lo3 = 0, hi3 = 0;
        bool fresh = false;
        bool resum_exit = false;  // left after the sums had moved on: re-sum, then advance
#pragma unroll 1
        for (;;) {
            const int m = s.m;
            const int n_in = s.lo_m - s.lo2, lv = max(s.hi2, s.lo_m), n_out = s.hi - lv;
            const bool fresh0 = (s.hi2 <= s.lo_m) || (s.hi2 == s.lo2);
            const float sh = (float)(s.t_ref - (int)t0_of(g, m - 1));
            const bool calm = has_edge && m != m_beg && !fresh0 && n_in <= 1 && n_out <= 1 &&
                              !(sh * kexp < kReanchorArg) && s.hi - s.lo_m >= pr.min_atoms;
            if (!__all_sync(kFull, calm)) break;
            const int a_in = min(s.lo2, a_last), a_out = min(lv, a_last);
            if ((unsigned)(a_in - in_base) >= 32u) {  // warp-uniform: stage the next 32 entering atoms
                in_base = max(a_in - 31, 0);
                const int al = min(in_base + lane, a_last);
                __syncwarp();
                s_tin[warp][lane] = __ldg(bd.t + al);
#pragma unroll
                for (int q = 0; q < TPC; ++q)
                    ldg_record(rec[q] + 2 * al, s_in[warp][q][2 * lane], s_in[warp][q][2 * lane + 1]);
                __syncwarp();
            }
            // -- record of the leaving atom, indices of the next step
            const int t_out = ldg_int_now(bd.t + a_out);
            ulonglong2 oa[TPC], ob[TPC];
#pragma unroll
            for (int q = 0; q < TPC; ++q) ldg_record_now(rec[q] + 2 * a_out, oa[q], ob[q]);
            lo3 = s.lo2, hi3 = s.hi2;
            if (m - 1 > m_beg) {
                lo3 = __ldg(bd.lo + m - 2);
                hi3 = max(__ldg(bd.edge + (jn + (m - 2) * bd.e_m)), lo3);
            }
            // -- a4: eq. (7) in fp32 for the TPC templates, one vote on "all well conditioned"
            float twoF[TPC];
            bool bad = false;
#pragma unroll
            for (int q = 0; q < TPC; ++q) {
                float A, B, far, fai, fbr, fbi;
                unpack2(s.acc[q].ab, A, B);
                unpack2(s.acc[q].fa, far, fai);
                unpack2(s.acc[q].fb, fbr, fbi);
                const float C = s.acc[q].c;
                const float p = A * B;
                const float D = fmaf(-C, C, p);
                const float na = fmaf(far, far, fai * fai);
                const float nb = fmaf(fbr, fbr, fbi * fbi);
                const float re = fmaf(far, fbr, fai * fbi);
                float num = B * na;
                num = fmaf(A, nb, num);
                num = fmaf(-2.0f * C, re, num);
                twoF[q] = 2.0f * num * rcp_approx_s(D);
                // (no short-circuit: four compares into one predicate)
                const bool ok = (D > 0.015625f * p) & (p > 1.0e-30f) & (p < 1.0e30f) &
                                (fabsf(twoF[q]) < 3.0e38f);
                bad = bad | !ok;
            }
            if (__any_sync(kFull, bad)) break;
            {
                // -- a5, branch-free
                if (pr.out_maps) {  // (uniform; a search stores no maps)
#pragma unroll
                    for (int q = 0; q < TPC; ++q)
                        if (n_ok && tpl0 + q < pr.n_templates) {
                            const int64_t o = ((int64_t)(tpl0 + q) * g.N_t0 + m) * g.N_tau + n;
                            pr.out_maps[o] = twoF[q];
                            if (pr.out_flags) pr.out_flags[o] = (uint8_t)0;
                        }
                }
                float x[TPC];
                bool move = false;
#pragma unroll
                for (int q = 0; q < TPC; ++q) {
                    const bool better = twoF[q] >= s.mg_best[q];
                    s.mg_best[q] = better ? twoF[q] : s.mg_best[q];
                    s.mg_m[q] = better ? m : s.mg_m[q];
                    x[q] = fmaf(twoF[q], kHalfLog2eS, -s.mg_ref2[q]);
                    move = move | (x[q] > 60.0f);
                }
                if (__any_sync(kFull, move)) {  // rare: move the reference of the log-sum-exp
#pragma unroll
                    for (int q = 0; q < TPC; ++q)
                        if (x[q] > 60.0f) {
                            s.mg_sum[q] *= ex2_approx(-x[q]);
                            s.mg_ref2[q] = twoF[q] * kHalfLog2eS;
                            x[q] = 0.0f;
                        }
                }
#pragma unroll
                for (int q = 0; q < TPC; ++q) s.mg_sum[q] += ex2_approx(x[q]);

                // -- the sums move on to cell m - 1
                const int t_in = s_tin[warp][a_in - in_base];
                const float e_in = ex2_approx((float)(t_in - s.t_ref) * kexp);
                const float e_out = ex2_approx((float)(t_out - s.t_ref) * kexp);
                fresh = false;
#pragma unroll
                for (int q = 0; q < TPC; ++q) {
                    const ulonglong2 ia = s_in[warp][q][2 * (a_in - in_base)];
                    const ulonglong2 ib = s_in[warp][q][2 * (a_in - in_base) + 1];
                    float dtc, ab;
                    unpack2(ia.x, dtc, ab);
                    // (fmaf(dtc, 0, e): NaN for an atom that is not finite, pack.cu; the select
                    // keeps an atom that is not part of this step out even then)
                    const float wi = n_in ? fmaf(dtc, 0.0f, e_in) : 0.0f;
                    acc_add(s.acc[q], wi, wi * wi, ia, ib);
                    unpack2(oa[q].x, dtc, ab);
                    const float wo = n_out ? -fmaf(dtc, 0.0f, e_out) : 0.0f;
                    acc_add(s.acc[q], wo, wo * fabsf(wo), oa[q], ob[q]);
                    float A, B;
                    unpack2(s.acc[q].ab, A, B);
                    s.A_max[q] = fmaxf(s.A_max[q], A);
                    fresh = fresh | !(A * kGuard >= s.A_max[q]);  // (see slide_step_generic)
                }
                if (STATS) {
                    s.n_term[1] += (unsigned)n_in;
                    s.n_term[2] += (unsigned)n_out;
                }
                if (__any_sync(kFull, fresh)) {  // rare: some lane's window lost its weight
                    resum_exit = true;
                    break;
                }
                s.m = m - 1;
                s.lo_m = s.lo2;
                s.hi = s.hi2;
                s.lo2 = lo3;
                s.hi2 = hi3;
            }
        }
        // ---- cold: what the fast path left undone
        const SlideCtx c = {packed, n_pad, tpl0, n, n_ok ? 1 : 0, m_beg, kexp};
        SlideState<TPC> tmp;
        if (resum_exit) {
            if (fresh) {
                slide_copy<TPC>(tmp, s);
                slide_resum<TPC, STATS>(tmp, pr, c);
                slide_copy<TPC>(s, tmp);
            }
            s.m -= 1;
            s.lo_m = s.lo2;
            s.hi = s.hi2;
            s.lo2 = lo3;
            s.hi2 = hi3;
        } else {
            slide_copy<TPC>(tmp, s);
            finished = slide_step_generic<TPC, STATS>(tmp, pr, c);
            slide_copy<TPC>(s, tmp);
        }
    }
    const int n_visited = warp * 32 < n_count ? m_end - m_beg : 0;
    if (STATS) {
        // (terms of out-of-range tau slots and of ragged template groups were not summed for real)
        unsigned long long v[5];
        const unsigned long long ntpl = n_ok ? (unsigned long long)min(TPC, pr.n_templates - tpl0) : 0ull;
#pragma unroll
        for (int i = 0; i < 4; ++i) v[i] = (unsigned long long)s.n_term[i] * ntpl;
        v[4] = (unsigned long long)n_visited * ntpl;
#pragma unroll
        for (int i = 1; i < 5; ++i) {
#pragma unroll
            for (int sft = 16; sft >= 1; sft >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], sft);
            if (lane == 0 && v[i]) atomicAdd(stats + i, v[i]);
        }
    }
    if (partials) {
#pragma unroll
        for (int q = 0; q < TPC; ++q) {
            Marg a;
            marg_init(a);
            const int nv = n_visited - s.n_bad[q];
            if (n_ok && nv > 0) {
                a.best = s.mg_best[q];
                a.idx = s.mg_m[q] * g.N_tau + n;
                a.M = 0.5f * s.mg_best[q];
                a.S = s.mg_sum[q] * ex2_approx(s.mg_ref2[q] - s.mg_best[q] * kHalfLog2eS);
                a.nvalid = nv;
            }
            __syncthreads();  // s_red is reused (by the next template, the next pass)
            marg_block_reduce<NT>(a, s_red);
            if (threadIdx.x == 0 && tpl0 + q < pr.n_templates)
                partial_store(partials + ((int64_t)(tpl0 + q) * n_segs + seg) * n_nblocks + j, a);
        }
    }
}

// ---- the three kernels built from the two bodies ----------------------------------------------
template <int NT, int RT, int TPC, bool STATS>
__global__ void __launch_bounds__(NT, RT * TPC >= 8 ? 4 : 5)
    exp_window_kernel(const Problem pr, const ulonglong2 *__restrict__ packed, const int n_pad,
                      float4 *__restrict__ W0, const int n_nblocks, const int n_segs,
                      const int seg_len, const int n_limit, unsigned long long *__restrict__ stats)
{
    exp_window_body<NT, RT, TPC, STATS>(pr, packed, n_pad, W0, blockIdx.x, n_nblocks, n_segs, seg_len,
                                        n_limit, stats);
}

template <int NT, int TPC, bool STATS>
__global__ void __launch_bounds__(NT, NT == 128 ? (TPC == 1 ? 5 : TPC == 2 ? 4 : 3) : 1)
    exp_slide_kernel(const __grid_constant__ Problem pr, const ulonglong2 *__restrict__ packed,
                     const int n_pad,
                     const float4 *__restrict__ W0, Partial *__restrict__ partials,
                     const int n_nblocks, const int n_segs, const int seg_len,
                     unsigned long long *__restrict__ stats)
{
    exp_slide_body<NT, TPC, STATS>(pr, packed, n_pad, W0, partials, blockIdx.x, n_nblocks, n_segs,
                                   seg_len, stats);
}

// Also measured (B200, config 4 x 2048 templates, with the slide loop of that time): both phases
// in ONE kernel (a CTA sums the windows of its 512 tau values, then slides them in four passes),
// hoping that CTAs in different phases overlap the FP32-bound window sums with the latency-bound
// sliding: 4.53 ms against 4.10 ms for the two kernels back to back (128 registers with spills,
// 16 warps per SM for both phases).  The two kernels take 2.06 + 1.15 ms now.

template <int NT, int TPC>
cudaError_t launch_tpc(const Plan &pl, const Problem &pr, const ulonglong2 *packed,
                       const float4 *W0, Partial *partials, cudaStream_t st)
{
    const int64_t groups = (pl.n_templates + TPC - 1) / TPC;
    const int64_t n_ctas = (int64_t)pl.n_nblocks * pl.n_segs * groups;
    if (pl.stats)
        return launch_k(exp_slide_kernel<NT, TPC, true>, (unsigned)n_ctas, NT, 0, st, pr, packed,
                          pl.n_pad, W0, partials, pl.n_nblocks, pl.n_segs, pl.seg_len, pl.stats);
    return launch_k(exp_slide_kernel<NT, TPC, false>, (unsigned)n_ctas, NT, 0, st, pr, packed,
                      pl.n_pad, W0, partials, pl.n_nblocks, pl.n_segs, pl.seg_len, pl.stats);
}

template <int NT>
cudaError_t launch_nt(const Plan &pl, const Problem &pr, const ulonglong2 *packed,
                      const float4 *W0, Partial *partials, cudaStream_t st)
{
    if (pl.slide_tpc == 4 && NT == 128) return launch_tpc<128, 4>(pl, pr, packed, W0, partials, st);
    if (pl.slide_tpc == 2) return launch_tpc<NT, 2>(pl, pr, packed, W0, partials, st);
    return launch_tpc<NT, 1>(pl, pr, packed, W0, partials, st);
}

// window sums: RT tau values per thread x TPC templates per CTA
template <int NT, int RT, int TPC>
cudaError_t launch_win(const Plan &pl, const Problem &pr, const ulonglong2 *packed, float4 *W0,
                       cudaStream_t st)
{
    const int n_limit = pl.mom_n16;  // tau indices below the moment kernel's regions
    if (n_limit <= 0) return cudaSuccess;
    const int nblk = (n_limit + NT * RT - 1) / (NT * RT);
    const int64_t groups = (pl.n_templates + TPC - 1) / TPC;
    const int64_t n_ctas = (int64_t)nblk * pl.n_segs * groups;
    if (pl.stats)
        return launch_k(exp_window_kernel<NT, RT, TPC, true>, (unsigned)n_ctas, NT, 0, st, pr,
                          packed, pl.n_pad, W0, nblk, pl.n_segs, pl.seg_len, n_limit, pl.stats);
    return launch_k(exp_window_kernel<NT, RT, TPC, false>, (unsigned)n_ctas, NT, 0, st, pr,
                      packed, pl.n_pad, W0, nblk, pl.n_segs, pl.seg_len, n_limit, pl.stats);
}

// window sums of the tau indices [mom_n16, N_tau) in groups of 16, 32 and 64 (exp_moment_kernel)
cudaError_t launch_mom(const Plan &pl, const Problem &pr, const ulonglong2 *packed, float4 *W0,
                       cudaStream_t st)
{
    const int G64 = (pl.grid.N_tau - pl.mom_n64 + 63) / 64, G32 = (pl.mom_n64 - pl.mom_n32 + 31) / 32,
              G16 = (pl.mom_n32 - pl.mom_n16 + 15) / 16;
    if (G64 + G32 + G16 <= 0) return cudaSuccess;
    const int n_gblocks = (G64 + G32 + G16 + kMomGW - 1) / kMomGW;
    const int64_t quads = (pl.n_templates + 3) / 4;
    const int64_t n_ctas = (int64_t)n_gblocks * pl.n_segs * quads;
    if (pl.stats)
        return launch_k(exp_moment_kernel<true>, (unsigned)n_ctas, 32 * kMomNW, 0, st, pr, packed,
                          pl.n_pad, W0, pl.mom_n16, pl.mom_n32, pl.mom_n64, n_gblocks, pl.n_segs, pl.seg_len,
                          pl.stats);
    return launch_k(exp_moment_kernel<false>, (unsigned)n_ctas, 32 * kMomNW, 0, st, pr, packed,
                      pl.n_pad, W0, pl.mom_n16, pl.mom_n32, pl.mom_n64, n_gblocks, pl.n_segs, pl.seg_len, pl.stats);
}

}  // namespace

cudaError_t launch_exp_scan(const Plan &pl, const Problem &pr, const void *packed, void *w0,
                            Partial *partials, cudaStream_t st)
{
    const ulonglong2 *rec = static_cast<const ulonglong2 *>(packed);
    float4 *W0 = static_cast<float4 *>(w0);
    cudaError_t e;
    switch ((pl.win_nt == 64 ? 100 : 0) + pl.win_rt * 10 + pl.win_tpc) {
    case 42: e = launch_win<128, 4, 2>(pl, pr, rec, W0, st); break;
    case 41: e = launch_win<128, 4, 1>(pl, pr, rec, W0, st); break;
    case 22: e = launch_win<128, 2, 2>(pl, pr, rec, W0, st); break;
    case 21: e = launch_win<128, 2, 1>(pl, pr, rec, W0, st); break;
    case 142: e = launch_win<64, 4, 2>(pl, pr, rec, W0, st); break;
    case 141: e = launch_win<64, 4, 1>(pl, pr, rec, W0, st); break;
    case 122: e = launch_win<64, 2, 2>(pl, pr, rec, W0, st); break;
    case 121: e = launch_win<64, 2, 1>(pl, pr, rec, W0, st); break;
    case 112:
    case 12: e = launch_win<64, 1, 2>(pl, pr, rec, W0, st); break;
    default: e = launch_win<64, 1, 1>(pl, pr, rec, W0, st); break;
    }
    if (e != cudaSuccess) return e;
    e = launch_mom(pl, pr, rec, W0, st);
    if (e != cudaSuccess) return e;
    switch (pl.tile.NT) {
    case 128: return launch_nt<128>(pl, pr, rec, W0, partials, st);
    case 64: return launch_nt<64>(pl, pr, rec, W0, partials, st);
    case 32: return launch_nt<32>(pl, pr, rec, W0, partials, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace tfstat
