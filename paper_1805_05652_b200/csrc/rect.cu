// rect.cu -- steps a2 + a4 + a5 for the rectangular window (eq. 3).
//
// The paper keeps running partial sums over tau per t0 with N_t0 workers.  Here:
//
//  1. rect_scan_kernel, scan blocks: exclusive prefix sums P of the 7 atom channels in fp64,
//     1024 atoms per CTA, block totals exchanged through flags inside the launch (an fp32 prefix
//     over a year of atoms cancels catastrophically for short windows far from the origin,
//     SURVEY.md H1; fp64 differences of fp32 data are exact to ~1e-13).
//  2. rect_scan_kernel, step blocks (same launch): every window end t0_m + tau_n lies on the
//     edge lattice (bounds.cu), so the atoms that ENTER a window when tau grows by TWO grid
//     steps are the same for every cell with the same lattice point j:
//     H[j] = P[edge[j + 2 e_n]] - P[edge[j]], rounded once to fp32 (a sum of a few atoms: exact
//     to 2^-24 of its own size).  The table K[j] = (H[j], H[j + e_n]) holds them as channel
//     pairs, 64 bytes per lattice point, planar so that a warp reads whole 128-byte lines.
//  3. rect_run_kernel: one thread walks one t0 row along tau, two columns at a time: its state
//     is the seven sums of columns (n, n+1) as packed fp32x2 pairs.  It starts each column tile
//     from the exact window sums P[hi] - P[lo] and then only ADDS K -- the paper's running sum,
//     with pre-aggregated steps -- so two cells cost 8 packed adds + 13 packed multiply-adds +
//     2 MUFU.RCP (eq. 7, pair_closure).  Row m + 2 e_n / e_m uses the same K entries one
//     pair-step later, so a thread owns Q = 2 such rows and keeps a sliding register window of
//     K: 16 bytes of L1 traffic per cell; the other row groups of its CTA find them in L1.  The
//     closure runs in fp32 where the cell is well conditioned (D > AB/64, error <= ~1e-4
//     relative); groups with any other cell, and the leading columns that hold fewer than
//     min_atoms atoms, are recomputed in fp64 from P.  2F values are transposed through
//     (swizzled) shared memory (thread = row, but the map is tau-fastest) and leave as 64-byte
//     row segments.
//
//  3'. rect_tile_kernel (further down), instead of 2. and 3. where the lattice steps are small
//     (dt0 and dtau within a factor 4 of each other: the full-resolution grids): the direct form
//     S(m, n) = P[hi] - P[lo_m] tile by tile, as Phi[j] + U[m] with both terms staged once per
//     tile relative to an anchor atom -- no running sum, no dependency between cells, two cells
//     that share a lattice point per packed instruction, plain coalesced stores.
//
// Grids without an edge lattice (J = 0) or with very few t0 rows use the per-cell kernel
// rect_cells_kernel: S(m,n) = P[hi(m,n)] - P[lo(m)], closure in fp64.  Small problems take
// rect_small_kernel: everything in one launch, one CTA per template.
#include <algorithm>

#include "plan.h"

namespace tfstat {

namespace {

constexpr int kScanNT = 256;
constexpr int kScanPer = 4;                       // atoms per thread
constexpr int kScanBlock = kScanNT * kScanPer;    // atoms per CTA

// ---------------------------------------------------------------------------------------
// rect_scan_kernel: ONE launch builds the fp64 prefix P and the fp32 lattice steps G.
//
//  * scan blocks (blockIdx < n_scan): kScanBlock atoms each.  A block publishes the totals of
//    its 7 channels (agg + ready flag) BEFORE it waits for anybody, then sums the totals of
//    the blocks in front of it, scans its own atoms and writes P (done flag).  Blocks only wait
//    for lower blockIdx, which the hardware dispatches first, so the wait cannot deadlock.
//  * step blocks (blockIdx >= n_scan): 256 lattice points each; a thread waits for the scan
//    blocks that own its two P entries, then G[j] = P[edge[j + e_n]] - P[edge[j]].
//  Flags are zeroed by bounds_kernel (or a memset) before the launch.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ void st_release(int32_t *p, const int32_t v)
{
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// Wait for two flags: poll with relaxed loads and a back-off (an acquire load per poll
// invalidates the whole L1 and starves the producers of issue slots), then ONE acquire fence.
__device__ __forceinline__ void wait_flags2(const int32_t *p, const int32_t *q)
{
    int32_t v, w;
    for (;;) {
        asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
        asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(w) : "l"(q) : "memory");
        if (v != 0 && w != 0) break;
        __nanosleep(64);
    }
    asm volatile("fence.acq_rel.gpu;" ::: "memory");
}

// window sums of atoms [lo, hi) from the prefix, in fp64; L2 loads (P may have been written by
// another SM during this very launch)
__device__ __forceinline__ Sums64 prefix_diff_cg(const double2 *P, const int lo, const int hi)
{
    const double2 l0 = __ldcg(P + (int64_t)lo * 4), l1 = __ldcg(P + (int64_t)lo * 4 + 1),
                  l2 = __ldcg(P + (int64_t)lo * 4 + 2), l3 = __ldcg(P + (int64_t)lo * 4 + 3);
    const double2 h0 = __ldcg(P + (int64_t)hi * 4), h1 = __ldcg(P + (int64_t)hi * 4 + 1),
                  h2 = __ldcg(P + (int64_t)hi * 4 + 2), h3 = __ldcg(P + (int64_t)hi * 4 + 3);
    Sums64 s;
    s.A = h0.x - l0.x;
    s.B = h0.y - l0.y;
    s.C = h1.x - l1.x;
    s.far = h1.y - l1.y;
    s.fai = h2.x - l2.x;
    s.fbr = h2.y - l2.y;
    s.fbi = h3.x - l3.x;
    if (h3.y - l3.y > 0.5) s.A = nan("");  // the window holds a non-finite atom: D <= 0 flag
    return s;
}

// The running Fa, Fb sums are carried scaled by sqrt(2), so eq. (7) on them yields 2F directly.
constexpr double kSqrt2 = 1.41421356237309504880;
constexpr int kStepSplit = 4;                    // threads per lattice point (step role)
constexpr int kStepPts = kScanNT / kStepSplit;   // lattice points per step CTA
constexpr int kDirectStep = 64;    // lattice steps of at most this many atoms are summed directly

// P[tpl][i][ch], i = 0..n_atoms, ch = 0..7 (7 used): 64 B per entry.
// K[tpl][q][j], q = 0..3, j = 0..J, 16 B per element (64 B per lattice point): the channel pairs (x of H[j], x of H[j + e_n]) for
// x = A, B | C, Re Fa | Im Fa, Re Fb | Im Fb, -C (Fa, Fb scaled by sqrt 2); entry J is all zero
// (out-of-range reads of the running kernel are clamped to it).  -C comes last so that a running
// kernel that reads K from global memory can leave it out (see load_k).
__global__ void __launch_bounds__(kScanNT)
    rect_scan_kernel(const Problem pr, double *__restrict__ agg, int32_t *__restrict__ flags,
                     double *__restrict__ prefix, ulonglong2 *__restrict__ K, const int nblk,
                     const int n_scan, const int steps_per_template)
{
    __shared__ double s_off[8];
    __shared__ double s_w[8][kScanNT / 32];
    const Bounds &bd = pr.bounds;
    const int N = bd.n_atoms;
    int32_t *ready = flags, *done = flags + n_scan;

    if ((int)blockIdx.x >= n_scan) {  // ---- step role ------------------------------------
        // kStepSplit threads per lattice point j share the sum H[j] of the atoms in
        // [edge[j], edge[j + 2 e_n]): what a row gains when it moves on by two columns.  H[j] is
        // the first half of the pairs of K[j] and the second half of the pairs of K[j - e_n].
        const int sb = blockIdx.x - n_scan;
        const int tpl = sb / steps_per_template;
        const int j = (sb % steps_per_template) * kStepPts + (int)threadIdx.x / kStepSplit;
        const int sub = threadIdx.x % kStepSplit;
        // the kStepSplit lanes of a lattice point branch together, the warp need not
        const unsigned grp_mask = ((1u << kStepSplit) - 1u) << ((threadIdx.x & 31) - sub);
        const int64_t jb = (int64_t)j + 2 * (int64_t)bd.e_n;
        const bool in_lattice = jb < bd.J;  // beyond: only cells outside the map would use it
        double acc[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        int a = 0, b = 0;
        if (in_lattice) {
            a = __ldg(bd.edge + j);
            b = __ldg(bd.edge + jb);
        }
        if (b - a <= kDirectStep) {
            // short step: sum its atoms directly (fp64), independent of the scan blocks
            const float *__restrict__ base = pr.atoms + (int64_t)tpl * pr.template_stride;
#pragma unroll 2
            for (int al = a + sub; al < b; al += kStepSplit) {
#pragma unroll
                for (int ch = 0; ch < 7; ++ch) acc[ch] += (double)__ldg(base + ch * pr.ld + al);
            }
#pragma unroll
            for (int ch = 0; ch < 7; ++ch)
#pragma unroll
                for (int sh = 1; sh < kStepSplit; sh <<= 1)
                    acc[ch] += __shfl_xor_sync(grp_mask, acc[ch], sh);
        } else {  // whole groups of kStepSplit lanes take this branch together
            const int32_t *da = done + tpl * nblk + max(a - 1, 0) / kScanBlock;
            const int32_t *db = done + tpl * nblk + max(b - 1, 0) / kScanBlock;
            wait_flags2(db, da);  // scan blocks finish roughly in order: the later one first
            const double2 *P =
                reinterpret_cast<const double2 *>(prefix + (int64_t)tpl * (N + 1) * 8);
            const Sums64 h = prefix_diff_cg(P, a, b);
            acc[0] = h.A;
            acc[1] = h.B;
            acc[2] = h.C;
            acc[3] = h.far;
            acc[4] = h.fai;
            acc[5] = h.fbr;
            acc[6] = h.fbi;
        }
        if (sub != 0 || j > bd.J) return;
        // planar: plane q of template tpl holds J + 1 16-byte elements, so that the lanes of a
        // warp (consecutive rows = consecutive j) read consecutive 16-byte words
        const int64_t pl = (int64_t)bd.J + 1;
        float *__restrict__ kf = reinterpret_cast<float *>(K + (int64_t)tpl * 4 * pl);
        const float v[8] = {(float)acc[0], (float)acc[1], (float)acc[2],
                            (float)(kSqrt2 * acc[3]), (float)(kSqrt2 * acc[4]),
                            (float)(kSqrt2 * acc[5]), (float)(kSqrt2 * acc[6]), (float)-acc[2]};
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            // channel c lives in plane c / 2, 8-byte pair c % 2 of the 16-byte element
            float *__restrict__ e = kf + ((int64_t)(c >> 1) * pl) * 4 + (c & 1) * 2;
            e[(int64_t)j * 4] = v[c];                                // first of the pair of K[j]
            if (j >= bd.e_n) e[((int64_t)j - bd.e_n) * 4 + 1] = v[c];  // second of K[j - e_n]
            // K[j]'s second halves for j > J - e_n belong to H beyond the lattice: zero
            if (j + bd.e_n > bd.J) e[(int64_t)j * 4 + 1] = 0.0f;
        }
        return;
    }

    // ---- scan role --------------------------------------------------------------------------
    const int tpl = blockIdx.x / nblk, blk = blockIdx.x % nblk;
    const float *__restrict__ base = pr.atoms + (int64_t)tpl * pr.template_stride;
    double *__restrict__ P = prefix + (int64_t)tpl * (N + 1) * 8;
    const int a0 = blk * kScanBlock + (int)threadIdx.x * kScanPer;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    // channel 7 counts the atoms that are not finite (a bad SFT): they enter the prefix as zeros
    // plus a count, so that only the windows that hold one are spoiled (prefix_diff), not every
    // window behind it
    float x[8][kScanPer];
#pragma unroll
    for (int ch = 0; ch < 7; ++ch)
#pragma unroll
        for (int i = 0; i < kScanPer; ++i)
            x[ch][i] = (a0 + i < N) ? __ldg(base + ch * pr.ld + a0 + i) : 0.0f;
#pragma unroll
    for (int i = 0; i < kScanPer; ++i) {
        bool bad = false;
#pragma unroll
        for (int ch = 0; ch < 7; ++ch) bad = bad || !(fabsf(x[ch][i]) < INFINITY);
        x[7][i] = bad ? 1.0f : 0.0f;
        if (bad) {
#pragma unroll
            for (int ch = 0; ch < 7; ++ch) x[ch][i] = 0.0f;
        }
    }

    double incl[8], tsum[8];
#pragma unroll
    for (int ch = 0; ch < 8; ++ch) {
        double t = 0.0;
#pragma unroll
        for (int i = 0; i < kScanPer; ++i) t += (double)x[ch][i];
        tsum[ch] = t;
#pragma unroll
        for (int sh = 1; sh < 32; sh <<= 1) {
            const double up = __shfl_up_sync(0xffffffffu, t, sh);
            if (lane >= sh) t += up;
        }
        incl[ch] = t;
        if (lane == 31) s_w[ch][warp] = t;
    }
    __syncthreads();
    {
        // publish this block's totals before waiting for anyone
        if (threadIdx.x < 32) {
            if (threadIdx.x < 8) {
                double t = 0.0;
#pragma unroll
                for (int w = 0; w < kScanNT / 32; ++w) t += s_w[threadIdx.x][w];
                __stcg(agg + (int64_t)blockIdx.x * 8 + threadIdx.x, t);
                __threadfence();
            }
            __syncwarp();
            if (threadIdx.x == 0) st_release(ready + blockIdx.x, 1);
        }
        // offset of this block: warp ch sums the totals of blocks [0, blk) of this template
        if (warp < 8) {
            // all lanes poll their flags together and the warp takes ONE acquire fence: a
            // wait_flag per lane would diverge and serialise up to 32 fences
            for (int b0 = 0; b0 < blk; b0 += 32) {
                const int b = b0 + lane;
                for (;;) {
                    int32_t v = 1;
                    if (b < blk)
                        asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];"
                                     : "=r"(v)
                                     : "l"(ready + tpl * nblk + b)
                                     : "memory");
                    if (__all_sync(0xffffffffu, v != 0)) break;
                    __nanosleep(32);
                }
            }
            asm volatile("fence.acq_rel.gpu;" ::: "memory");
            double t = 0.0;
            for (int b = lane; b < blk; b += 32)
                t += __ldcg(agg + ((int64_t)tpl * nblk + b) * 8 + warp);
#pragma unroll
            for (int sh = 16; sh >= 1; sh >>= 1) t += __shfl_xor_sync(0xffffffffu, t, sh);
            if (lane == 0) s_off[warp] = t;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0 && blk == 0) {
#pragma unroll
        for (int ch = 0; ch < 8; ++ch) P[ch] = 0.0;
    }
#pragma unroll
    for (int ch = 0; ch < 8; ++ch) {
        double run = s_off[ch] + incl[ch] - tsum[ch];
        for (int w = 0; w < warp; ++w) run += s_w[ch][w];
#pragma unroll
        for (int i = 0; i < kScanPer; ++i) {
            run += (double)x[ch][i];
            if (a0 + i < N) P[(int64_t)(a0 + i + 1) * 8 + ch] = run;
        }
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) st_release(done + blockIdx.x, 1);
}

// window sums of atoms [lo, hi) from the prefix, in fp64
__device__ __forceinline__ Sums64 prefix_diff(const double2 *__restrict__ P, const int lo,
                                              const int hi)
{
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
    if (h3.y - l3.y > 0.5) s.A = nan("");  // the window holds a non-finite atom: D <= 0 flag
    return s;
}

// ---------------------------------------------------------------------------------------
// generic per-cell kernel (no edge lattice / very few t0 rows)
// ---------------------------------------------------------------------------------------
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
        const Sums64 s = prefix_diff(P, lo, hi);
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

// ---------------------------------------------------------------------------------------
// small problems: everything in ONE launch, one CTA per template
//
// A call on a small map is otherwise a chain of four dependent launches (bounds, scan, cells,
// finalize) of ~5 us each whatever the size -- the "overhead-dominated" regime the paper
// reports for rectangular windows on GPUs.  Here a CTA stages the timestamps and
// the fp64 prefix sums of its template in shared memory (one warp per channel), finds lo / hi of
// every cell by binary search in shared memory, closes in fp64, reduces its marginals and
// writes the tfstat_result itself: BASELINE.json config 1 (24 x 24 cells, 48 atoms) in one
// launch, 1000 such templates in one wave.
// ---------------------------------------------------------------------------------------
constexpr int kSmallNT = 256;

__device__ __forceinline__ int lower_bound_s(const int32_t *s_t, const int n, const long long x)
{
    int a = 0, b = n;
    while (a < b) {
        const int mid = (a + b) >> 1;
        if ((long long)s_t[mid] < x) a = mid + 1;
        else b = mid;
    }
    return a;
}

__global__ void __launch_bounds__(kSmallNT)
    rect_small_kernel(const Problem pr)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ Marg s_red[32];
    const Grid g = pr.grid;
    const int N = pr.bounds.n_atoms;
    double *s_P = reinterpret_cast<double *>(smem_raw);              // [(N + 1)][8], 7 used
    int32_t *s_t = reinterpret_cast<int32_t *>(s_P + (size_t)(N + 1) * 8);  // [N]
    const int tpl = blockIdx.x;
    const float *__restrict__ base = pr.atoms + (int64_t)tpl * pr.template_stride;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    uint8_t *s_bad = reinterpret_cast<uint8_t *>(s_t + N);  // [N]: atom is not finite (bad SFT)
    for (int i = threadIdx.x; i < N; i += kSmallNT) {
        s_t[i] = __ldg(pr.bounds.t + i);
        bool bad = false;
#pragma unroll
        for (int ch = 0; ch < 7; ++ch) bad = bad || !(fabsf(__ldg(base + ch * pr.ld + i)) < INFINITY);
        s_bad[i] = bad ? 1 : 0;
    }
    __syncthreads();
    // a2: exclusive fp64 prefix of channel `warp`, 32 atoms per step of a warp-wide scan; bad
    // atoms enter as zeros and are counted in channel 7, so that they only spoil their own windows
    {
        const float *__restrict__ row = base + min(warp, 6) * pr.ld;
        double carry = 0.0;
        if (lane == 0) s_P[warp] = 0.0;
        for (int i0 = 0; i0 < N; i0 += 32) {
            const int i = i0 + lane;
            double v = 0.0;
            if (i < N) v = warp == 7 ? (double)s_bad[i] : s_bad[i] ? 0.0 : (double)__ldg(row + i);
#pragma unroll
            for (int sh = 1; sh < 32; sh <<= 1) {
                const double up = __shfl_up_sync(0xffffffffu, v, sh);
                if (lane >= sh) v += up;
            }
            v += carry;
            if (i < N) s_P[(size_t)(i + 1) * 8 + warp] = v;
            carry = __shfl_sync(0xffffffffu, v, 31);
        }
    }
    __syncthreads();

    Marg mg;
    marg_init(mg);
    const int n_cells = g.N_t0 * g.N_tau;
    const int64_t map_base = (int64_t)tpl * n_cells;
    for (int i = threadIdx.x; i < n_cells; i += kSmallNT) {
        const int m = i / g.N_tau, n = i - m * g.N_tau;
        const long long t0 = t0_of(g, m);
        const int lo = lower_bound_s(s_t, N, t0);
        const int hi = lower_bound_s(s_t, N, t0 + tau_of(g, n));  // k = 1: rectangular
        const double *pl = s_P + (size_t)lo * 8, *ph = s_P + (size_t)hi * 8;
        Sums64 s;
        s.A = ph[0] - pl[0];
        s.B = ph[1] - pl[1];
        s.C = ph[2] - pl[2];
        s.far = ph[3] - pl[3];
        s.fai = ph[4] - pl[4];
        s.fbr = ph[5] - pl[5];
        s.fbi = ph[6] - pl[6];
        if (ph[7] - pl[7] > 0.5) s.A = nan("");  // the window holds a non-finite atom
        uint32_t fl;
        const float twoF = closure_2F(s, hi - lo, pr.min_atoms, fl);
        if (pr.out_maps) pr.out_maps[map_base + i] = twoF;
        if (pr.out_flags) pr.out_flags[map_base + i] = (uint8_t)fl;
        if (!fl) marg_add(mg, twoF, i);
    }
    if (pr.out) {
        marg_block_reduce<kSmallNT>(mg, s_red);
        if (threadIdx.x == 0) {
            tfstat_result r;
            r.n_valid = mg.nvalid;
            if (mg.nvalid > 0) {
                r.max2F = mg.best;
                r.m = mg.idx / g.N_tau;
                r.n = mg.idx % g.N_tau;
                r.logB = (float)((double)mg.M + log((double)mg.S));
            } else {
                r.max2F = 0.0f;
                r.m = -1;
                r.n = -1;
                r.logB = -INFINITY;
            }
            pr.out[tpl] = r;
        }
    }
}

// ---------------------------------------------------------------------------------------
// running-sum kernel
// ---------------------------------------------------------------------------------------
constexpr int kRunNT = 64;   // 2 warps per CTA: measured 5 % faster than 128 (cheaper transpose barrier)
constexpr int kChunk = 16;   // columns between two write-outs of the transposed tile
constexpr int kPitch = 16;   // floats per tile row; the four 16-byte column groups of row i are
                             // XOR-swizzled with (i >> 1) & 3: conflict-free STS.128 and LDS.128
constexpr int kFPitch = 5;   // 32-bit words per flag-tile row (16 flag bytes + pad)
constexpr int kKsMaxEntries = 320;  // 64 B each: at most 20 KB of K per CTA in shared memory
constexpr float kCondFast = 1.0f / 64.0f;  // fp32 closure only if D > kCondFast * A * B
constexpr float kTiny = 1.0e-30f;          // ... and D > kTiny
constexpr float kHalfLog2e = 0.72134752044448170368f;

__device__ __forceinline__ u64 fadd2(const u64 a, const u64 b)
{
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

__device__ __forceinline__ float rcp_approx(const float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ill-conditioned, short or empty cell (m, n): the plain way, in fp64 straight from the prefix.
// Returns (2F, flags) packed in one 64-bit register.
__device__ __noinline__ u64 rect_cell_slow(const double2 *__restrict__ P,
                                           const int32_t *__restrict__ lo_tab,
                                           const int32_t *__restrict__ edge, const int m,
                                           const int64_t j, const int min_atoms)
{
    const int lo = __ldg(lo_tab + m);
    const int hi = max(__ldg(edge + j), lo);
    const Sums64 s = prefix_diff(P, lo, hi);
    uint32_t f;
    const float twoF = closure_2F(s, hi - lo, min_atoms, f);
    return pack2(twoF, __uint_as_float(f));
}

struct RunMarg {
    float best;   // max 2F
    int32_t idx;  // its flat index
    float ref2;   // reference exponent (log2 units) of the running sum
    float sum;    // sum 2^(F log2e - ref2)
    int32_t nv;
};

// Row state of the running kernel: 8 channel pairs, each (column n, column n + 1):
//   0 A   1 B   2 C   3 -C   4 Re Fa   5 Im Fa   6 Re Fb   7 Im Fb      (Fa, Fb times sqrt 2)
// so eq. (7) for TWO cells is 13 packed fp32x2 operations and 2 MUFU.RCP:
//   D = A B + (-C) C;  2|Fa|^2, 2|Fb|^2, 2 Re(Fa conj Fb);  num = B 2|Fa|^2 + A 2|Fb|^2
//   + 2 (-C) 2Re;  2F = num / D.
// -C is carried as a channel of its own because fma.rn.f32x2 has no operand negation
// (recomputing -C = -1 x C after every step instead puts a multiply on the dependent chain and
// measured 2-4 % slower on the one-year map).
struct PairOut {
    u64 res;  // 2F of (column n, column n + 1), fp32 fast path
    u64 t;    // D - kCondFast A B of the two cells: the fast path holds where t > 0
};

__device__ __forceinline__ PairOut pair_closure(const u64 (&S)[8])
{
    const u64 p = fmul2(S[0], S[1]);
    u64 D = p;
    ffma2(D, S[3], S[2]);
    PairOut o;
    // t = D - kCondFast A B - kTiny: the fast path also needs D well inside the normal fp32
    // range (atoms scaled far down: rcp.approx.ftz of a subnormal D is inf)
    o.t = fadd2(D, pack2(-kTiny, -kTiny));
    ffma2(o.t, p, pack2(-kCondFast, -kCondFast));
    u64 na = fmul2(S[4], S[4]);
    ffma2(na, S[5], S[5]);
    u64 nb = fmul2(S[6], S[6]);
    ffma2(nb, S[7], S[7]);
    u64 re = fmul2(S[4], S[6]);
    ffma2(re, S[5], S[7]);
    u64 num = fmul2(S[1], na);
    ffma2(num, S[0], nb);
    ffma2(num, S[3], re);
    ffma2(num, S[3], re);
    // atoms scaled far up: rcp.approx.ftz of D > 2^126 is 0 and the numerator overflows; 0 x inf
    // = NaN poisons t whenever num * A B leaves the fp32 range (false alarms only cost the fp64 path)
    ffma2(o.t, fmul2(num, p), 0ull);
    float d0, d1;
    unpack2(D, d0, d1);
    o.res = fmul2(num, pack2(rcp_approx(d0), rcp_approx(d1)));
    return o;
}

// 16 warps per SM for Q = 2 (128 registers): measured on B200 against 12 (162 registers, no
// spill), 20 (96) and 24 (80, spilling) warps per SM, which are 13 % to 58 % slower on config 5
// (one row per thread: 8 CTAs per SM too -- 5 % faster than 10, 12 % faster than 12)
//
// KS: the K entries a CTA walks (a run of ks_cap lattice points at most, see launch_run) are
// copied to shared memory first.  A warp's LDG.128 of 32 consecutive 16-byte entries starts at
// any multiple of 16 bytes, so each quarter-warp straddles two 128-byte lines and the load costs
// 7 to 8 L1 wavefronts; the same LDS.128 costs 4.  ncu on the one-year map: L1 data-pipe
// wavefronts 75 % of peak before, the limiter of this kernel.
template <int Q, bool MARG, bool KS>
__global__ void __launch_bounds__(kRunNT, 8)
    rect_run_kernel(const Problem pr, const double *__restrict__ prefix,
                    const ulonglong2 *__restrict__ K, Partial *__restrict__ partials,
                    const int roff, const int R, const int seg_cols, const int n_rowtiles,
                    const int n_coltiles, const int vec_ok, const int ks_cap, const int ks_lg)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ Marg s_red[32];
    constexpr int nrows = Q * kRunNT;
    float *tile = reinterpret_cast<float *>(smem_raw);                     // [nrows][kPitch]
    int *s_rowm = reinterpret_cast<int *>(tile + (size_t)nrows * kPitch);  // [nrows]
    uint32_t *ftile = reinterpret_cast<uint32_t *>(s_rowm + nrows);        // [nrows][kFPitch]

    const Grid g = pr.grid;
    const Bounds &bd = pr.bounds;
    const int rowtile = blockIdx.x % n_rowtiles;
    const int coltile = (blockIdx.x / n_rowtiles) % n_coltiles;
    const int tpl = blockIdx.x / (n_rowtiles * n_coltiles);
    const int lt = threadIdx.x;
    // Rows come in groups of Q roff consecutive rows; a thread owns rows res, res + roff, ..
    // of one group.  A CTA is R consecutive residues x (kRunNT / R) consecutive groups: the
    // same residue of the NEXT group walks the same K entries 2 Q columns later, so the groups
    // of a CTA find them in L1.
    int mbase = rowtile * kRunNT + lt;
    if (Q > 1) {
        const int gpc = kRunNT / R;           // groups per CTA
        const int n_restiles = (roff + R - 1) / R;
        const int res = (rowtile % n_restiles) * R + lt % R;
        const int grp = (rowtile / n_restiles) * gpc + lt / R;
        mbase = res < roff ? grp * roff * Q + res : g.N_t0;  // ragged residue tile: no rows
    }
    const int n0 = coltile * seg_cols;
    const int n_end = min(n0 + seg_cols, g.N_tau);
    const double2 *__restrict__ P =
        reinterpret_cast<const double2 *>(prefix + (int64_t)tpl * (bd.n_atoms + 1) * 8);
    const ulonglong2 *__restrict__ k_t = K + (int64_t)tpl * (bd.J + 1) * 4;
    const int k_plane = bd.J + 1;
    // lattice points of this CTA: [jlo, jcap]; jcap = J (the zero entry) unless staged
    // Two rows per thread with roff = R = 2 or 4 (e_m = 1): the lanes of a warp read runs of R
    // entries 2 R apart, a 2-way bank conflict.  ks_lg = log2 R >= 0 stores the run in two halves,
    // the entries with an even (j / R) first: a warp is then on one half at every pair-step, on
    // 32 consecutive entries.
    const int ks_half = ks_cap >> 1;
    auto ks_pos = [&](const int j) -> int {
        if (ks_lg < 0) return j;
        return ((j >> ks_lg) & 1) * ks_half + ((j >> (ks_lg + 1)) << ks_lg) + (j & ((1 << ks_lg) - 1));
    };
    int jlo = 0, jcap = bd.J;
    ulonglong2 *ks = reinterpret_cast<ulonglong2 *>(
        smem_raw + (size_t)nrows * (kPitch * 4 + 4 + (pr.out_flags ? kFPitch * 4 : 0)));
    if (KS) {
        int mb_lo = rowtile * kRunNT;
        if (Q > 1) {
            const int gpc = kRunNT / R, n_restiles = (roff + R - 1) / R;
            mb_lo = (rowtile / n_restiles) * gpc * roff * Q + (rowtile % n_restiles) * R;
        }
        jlo = (int)min((int64_t)mb_lo * bd.e_m + (int64_t)n0 * bd.e_n, (int64_t)bd.J);
        jcap = (int)min((int64_t)jlo + ks_cap - 1, (int64_t)bd.J);
        const int ne = jcap - jlo + 1;
        // (a flat loop over 4 ne elements needs an integer division per element: 10 % of the
        // kernel's instructions on the one-year map, ncu source page)
        for (int j = lt; j < ne; j += kRunNT) {
            const ulonglong2 *__restrict__ e = k_t + jlo + j;
            ulonglong2 *d = ks + ks_pos(j);
            const ulonglong2 q0 = __ldg(e), q1 = __ldg(e + k_plane), q2 = __ldg(e + 2 * k_plane),
                             q3 = __ldg(e + 3 * k_plane);
            d[0] = q0, d[ks_cap] = q1, d[2 * ks_cap] = q2, d[3 * ks_cap] = q3;
        }
    }

    // ---- exact start of every row at columns n0, n0 + 1 -------------------------------------
    // Rows outside the grid carry a dummy, perfectly conditioned state so that they stay on
    // the fast path; nothing of theirs is stored.
    u64 S[Q][8];
    bool rvalid[Q];
    int n_first[Q];  // first column of the row with at least min_atoms atoms (n0 if none earlier)
    bool all_valid = true;
    int n_valid_rows = 0, n_slow_end = n0;
    const bool want_map = pr.out_maps != nullptr, want_flags = pr.out_flags != nullptr;
    const int64_t map_base = (int64_t)tpl * g.N_t0 * g.N_tau;
#pragma unroll
    for (int b = 0; b < Q; ++b) {
        const int m = min(mbase + b * roff, g.N_t0);
        bool valid = m < g.N_t0;
        const int mc = min(m, g.N_t0 - 1);
        const int lo = __ldg(bd.lo + mc);
        const int64_t j0 = (int64_t)mc * bd.e_m + (int64_t)n0 * bd.e_n;
        const int hi0 = max(__ldg(bd.edge + j0), lo);
        const int hi1 = max(__ldg(bd.edge + min(j0 + bd.e_n, (int64_t)bd.J - 1)), lo);
        const int cnt_end =
            max(__ldg(bd.edge + j0 + (int64_t)(n_end - 1 - n0) * bd.e_n), lo) - lo;
        // A row whose window still holds at most one atom (fewer than min_atoms) at the LAST
        // column of this tile is degenerate throughout: its cells are written here, directly,
        // and the row then runs as a dummy (rows at the end of the data or inside long gaps
        // would otherwise send every one of their cells through the fp64 path).
        if (valid && cnt_end <= 1 && cnt_end < pr.min_atoms) {
            uint32_t f1 = 3u;  // flags of a single-atom cell: bit 1 from the atom's own D in fp64
            if (cnt_end == 1) {
                const float *__restrict__ base = pr.atoms + (int64_t)tpl * pr.template_stride;
                const double a2 = (double)__ldg(base + lo), b2 = (double)__ldg(base + pr.ld + lo),
                             ab = (double)__ldg(base + 2 * pr.ld + lo);
                f1 = 1u | ((a2 * b2 - ab * ab > 0.0) ? 0u : 2u);
            }
            for (int n = n0; n < n_end; ++n) {
                const int64_t o = map_base + (int64_t)m * g.N_tau + n;
                if (want_map) pr.out_maps[o] = 0.0f;
                if (want_flags) {
                    const int c =
                        max(__ldg(bd.edge + j0 + (int64_t)(n - n0) * bd.e_n), lo) - lo;
                    pr.out_flags[o] = (uint8_t)(c == 0 ? 3u : f1);
                }
            }
            valid = false;
        }
        // columns [n0, n_ok) hold fewer than min_atoms atoms (counts grow with n): fp64 path
        int nk = n0;
        if (valid && hi0 - lo < pr.min_atoms) {
            int a = n0 + 1, e = n_end;  // first n in [a, e) with enough atoms, else n_end
            while (a < e) {
                const int mid = (a + e) >> 1;
                const int c = max(__ldg(bd.edge + j0 + (int64_t)(mid - n0) * bd.e_n), lo) - lo;
                if (c < pr.min_atoms) a = mid + 1;
                else e = mid;
            }
            nk = a;
        }
        n_first[b] = nk;
        n_slow_end = max(n_slow_end, nk);
        const Sums64 s0 = prefix_diff(P, lo, hi0), s1 = prefix_diff(P, lo, hi1);
        if (valid) {
            S[b][0] = pack2((float)s0.A, (float)s1.A);
            S[b][1] = pack2((float)s0.B, (float)s1.B);
            S[b][2] = pack2((float)s0.C, (float)s1.C);
            S[b][3] = pack2((float)-s0.C, (float)-s1.C);
            S[b][4] = pack2((float)(kSqrt2 * s0.far), (float)(kSqrt2 * s1.far));
            S[b][5] = pack2((float)(kSqrt2 * s0.fai), (float)(kSqrt2 * s1.fai));
            S[b][6] = pack2((float)(kSqrt2 * s0.fbr), (float)(kSqrt2 * s1.fbr));
            S[b][7] = pack2((float)(kSqrt2 * s0.fbi), (float)(kSqrt2 * s1.fbi));
        } else {
            S[b][0] = S[b][1] = pack2(1.0e15f, 1.0e15f);
#pragma unroll
            for (int ch = 2; ch < 8; ++ch) S[b][ch] = 0ull;
        }
        rvalid[b] = valid;
        all_valid = all_valid && valid;
        n_valid_rows += valid ? 1 : 0;
        s_rowm[b * kRunNT + lt] = valid ? m * g.N_tau : -1;  // element offset of the row
    }

    // ---- sliding window of K: slot i % Q holds pair-step i of row 0; row b is b steps ahead
    // (row m + b roff at column n sits on the lattice point of row m at column n + 2 b).  A
    // slot is refilled right after row 0 has used it, one whole pair-step of the other rows
    // before its next use, which hides the L1/L2 latency of the load.
    constexpr int NS = Q == 1 ? 2 : Q;
    u64 W[NS][8];
    // 32-bit lattice index (J <= 2^22); reads beyond the lattice are clamped to the zero entry J
    const int jstep = 2 * bd.e_n;
    int jw = (int)min((int64_t)mbase * bd.e_m + (int64_t)n0 * bd.e_n, (int64_t)jcap);
    if (KS) __syncthreads();
    auto load_k = [&](u64(&w)[8]) {
        ulonglong2 q0, q1, q2, q3;
        if (KS) {
            const ulonglong2 *e = ks + ks_pos(jw - jlo);
            q0 = e[0], q1 = e[ks_cap], q2 = e[2 * ks_cap], q3 = e[3 * ks_cap];
        } else {
            const ulonglong2 *__restrict__ e = k_t + jw;
            q0 = __ldg(e), q1 = __ldg(e + k_plane), q2 = __ldg(e + 2 * k_plane),
            // 8 of the 16 bytes: the increment of -C is that of C with both sign bits flipped
            // (two integer-pipe operations instead of 8 bytes through L1; config 5: 4-7 % faster.
            // From shared memory the same trade measured 2 % slower, so KS loads all 64 bytes.)
            q3.x = __ldg(reinterpret_cast<const u64 *>(e + 3 * k_plane));
            q3.y = q1.x ^ 0x8000000080000000ull;
        }
        w[0] = q0.x;
        w[1] = q0.y;
        w[2] = q1.x;
        w[3] = q3.y;
        w[4] = q1.y;
        w[5] = q2.x;
        w[6] = q2.y;
        w[7] = q3.x;
        jw = min(jw + jstep, jcap);
    };
#pragma unroll
    for (int k = 0; k < NS; ++k) load_k(W[k]);

    RunMarg rm;
    rm.best = -INFINITY;
    rm.idx = 0x7fffffff;
    rm.ref2 = -INFINITY;
    rm.sum = 0.0f;
    rm.nv = 0;

#pragma unroll 1
    for (int n = n0; n < n_end; n += kChunk) {
        const int ncols = min(kChunk, n_end - n);
#pragma unroll 1
        for (int c4 = 0; c4 < kChunk; c4 += 4) {
            const int left = ncols - c4;  // columns of this group inside the map (may be <= 0)
            if (left <= 0) break;
            // ---- 2 pair-steps (4 columns) x Q rows, straight-line packed fp32; cells that
            // fail the conditioning test are only marked here and redone afterwards ----------
            float res[Q][4];
            bool fast = true;
#pragma unroll
            for (int s = 0; s < 2; ++s) {
#pragma unroll
                for (int b = 0; b < Q; ++b) {
                    const PairOut o = pair_closure(S[b]);
                    unpack2(o.res, res[b][2 * s], res[b][2 * s + 1]);
                    float t0, t1;
                    unpack2(o.t, t0, t1);
                    fast = fast && (t0 > 0.0f) && (t1 > 0.0f);
#pragma unroll
                    for (int ch = 0; ch < 8; ++ch)
                        S[b][ch] = fadd2(S[b][ch], W[(s + b) % NS][ch]);
                    if (b == 0) load_k(W[s % NS]);
                }
            }
            uint32_t fw[Q];
#pragma unroll
            for (int b = 0; b < Q; ++b) fw[b] = 0u;
            if (!fast || n + c4 < n_slow_end) {
                // rare (a few hundred warps per million cells): every cell of the group is
                // redone the plain way, in fp64 from the prefix sums
#pragma unroll
                for (int b = 0; b < Q; ++b) {
#pragma unroll
                    for (int s = 0; s < 4; ++s) {
                        if (s < left && rvalid[b]) {
                            const int m = mbase + b * roff;
                            const int64_t j =
                                (int64_t)m * bd.e_m + (int64_t)(n + c4 + s) * bd.e_n;
                            float twoF, flf;
                            unpack2(rect_cell_slow(P, bd.lo, bd.edge, m, j, pr.min_atoms), twoF,
                                    flf);
                            res[b][s] = twoF;
                            fw[b] |= __float_as_uint(flf) << (8 * s);
                        }
                    }
                }
            }
#pragma unroll
            for (int b = 0; b < Q; ++b) {
                if (want_map)
                    *reinterpret_cast<float4 *>(tile + (size_t)(b * kRunNT + lt) * kPitch +
                                                4 * ((c4 >> 2) ^ ((lt >> 1) & 3))) =
                        make_float4(res[b][0], res[b][1], res[b][2], res[b][3]);
                if (want_flags) ftile[(b * kRunNT + lt) * kFPitch + (c4 >> 2)] = fw[b];
            }
            if (MARG && n_valid_rows > 0) {
                uint32_t any_fl = 0u;
#pragma unroll
                for (int b = 0; b < Q; ++b) any_fl |= fw[b];
                int n_ok = 4 * n_valid_rows;
                // cells outside the map (rows beyond N_t0, degenerate rows, columns beyond
                // N_tau) and flagged cells become -inf: they lose every max and add
                // exp(-inf) = 0
                if (any_fl != 0u || !all_valid || left < 4) {
                    n_ok = 0;
#pragma unroll
                    for (int b = 0; b < Q; ++b)
#pragma unroll
                        for (int s = 0; s < 4; ++s) {
                            if (!rvalid[b] || s >= left || ((fw[b] >> (8 * s)) & 0xffu) != 0u)
                                res[b][s] = -INFINITY;
                            else
                                n_ok += 1;
                        }
                }
                if (n_ok > 0) {
                    float gmax = res[0][0];
#pragma unroll
                    for (int b = 0; b < Q; ++b)
#pragma unroll
                        for (int s = 0; s < 4; ++s) gmax = fmaxf(gmax, res[b][s]);
                    if (gmax > rm.best) {  // rare: first cell of the group, in flat order
                        bool found = false;
#pragma unroll
                        for (int b = 0; b < Q; ++b)
#pragma unroll
                            for (int s = 0; s < 4; ++s)
                                if (!found && res[b][s] == gmax) {
                                    found = true;
                                    rm.idx = (mbase + b * roff) * g.N_tau + n + c4 + s;
                                }
                        rm.best = gmax;
                    }
                    if (fmaf(gmax, kHalfLog2e, -rm.ref2) > 60.0f) {  // rare: move the reference
                        rm.sum *= ex2_approx(rm.ref2 - gmax * kHalfLog2e);
                        rm.ref2 = gmax * kHalfLog2e;
                    }
                    float acc = 0.0f;
#pragma unroll
                    for (int b = 0; b < Q; ++b)
#pragma unroll
                        for (int s = 0; s < 4; ++s)
                            acc += ex2_approx(fmaf(res[b][s], kHalfLog2e, -rm.ref2));
                    rm.sum += acc;
                    rm.nv += n_ok;
                }
            }
        }
        if (want_map && !want_flags && vec_ok && ncols == kChunk) {  // the common, lean case
            __syncthreads();
            // 4 threads write the 64 bytes of one row; kRunNT / 4 rows per pass, all with the
            // same (row >> 1) & 3, so the swizzled word of a thread is the same in every pass
            float *__restrict__ dst = pr.out_maps + map_base + n + 4 * (threadIdx.x & 3);
            const float4 *__restrict__ src = reinterpret_cast<const float4 *>(tile) +
                                             ((threadIdx.x & 3) ^ ((threadIdx.x >> 3) & 3));
#pragma unroll 4
            for (int row = threadIdx.x >> 2; row < nrows; row += kRunNT / 4) {
                const int off = s_rowm[row];
                const float4 v = src[row * (kPitch / 4)];
                if (off >= 0) __stcs(reinterpret_cast<float4 *>(dst + off), v);
            }
            __syncthreads();
        } else if ((want_map || want_flags) && vec_ok) {
            __syncthreads();
            const int q4 = threadIdx.x & 3;
            for (int row = threadIdx.x >> 2; row < nrows; row += kRunNT / 4) {
                const int off = s_rowm[row];
                if (off < 0) continue;
                const int64_t o = map_base + off + n + 4 * q4;
                const int left = ncols - 4 * q4;
                if (left <= 0) continue;
                if (want_map) {
                    const float4 v =
                        *reinterpret_cast<const float4 *>(tile + (size_t)row * kPitch +
                                                          4 * (q4 ^ ((row >> 1) & 3)));
                    if (vec_ok && left >= 4) {
                        __stcs(reinterpret_cast<float4 *>(pr.out_maps + o), v);
                    } else {
                        pr.out_maps[o] = v.x;
                        if (left > 1) pr.out_maps[o + 1] = v.y;
                        if (left > 2) pr.out_maps[o + 2] = v.z;
                        if (left > 3) pr.out_maps[o + 3] = v.w;
                    }
                }
                if (want_flags) {
                    const uint32_t f = ftile[row * kFPitch + q4];
                    if (vec_ok && left >= 4) {
                        *reinterpret_cast<uint32_t *>(pr.out_flags + o) = f;
                    } else {
                        pr.out_flags[o] = (uint8_t)(f & 0xffu);
                        if (left > 1) pr.out_flags[o + 1] = (uint8_t)((f >> 8) & 0xffu);
                        if (left > 2) pr.out_flags[o + 2] = (uint8_t)((f >> 16) & 0xffu);
                        if (left > 3) pr.out_flags[o + 3] = (uint8_t)(f >> 24);
                    }
                }
            }
            __syncthreads();
        } else if (want_map || want_flags) {
            // rows that are not 16-byte aligned (N_tau not a multiple of 4), ragged last chunk,
            // flags: 16 lanes write the 16 columns of one row, so a warp stores two runs of
            // 64 contiguous bytes (4 scalar stores per thread at a 16-byte stride cost four
            // times the L1 wavefronts and L2 sectors: one-year map 985 us, now see DESIGN 6.3)
            __syncthreads();
            const int c = threadIdx.x & 15;
            if (c < ncols) {
                const int gsel = c >> 2, w = c & 3;
                if (want_map && !want_flags) {
                    // the common case, kept short (ncu, one-year map with N_tau = 17519: the
                    // generic loop below made this write-out 39 % of the kernel's instructions).
                    // row = r0 + (kRunNT / 16) k: (row >> 1) & 3 takes two values in turn, so the
                    // two swizzled words of a thread are fixed and the offsets stay 32-bit
                    static_assert(kRunNT / 16 == 4, "swizzle period of the scalar write-out");
                    const int r0 = threadIdx.x >> 4;
                    const float *__restrict__ t0p =
                        tile + (size_t)r0 * kPitch + 4 * (gsel ^ ((r0 >> 1) & 3)) + w;
                    const float *__restrict__ t1p =
                        tile + (size_t)(r0 + 4) * kPitch + 4 * (gsel ^ (((r0 >> 1) + 2) & 3)) + w;
                    float *__restrict__ dstb = pr.out_maps + map_base + n + c;
#pragma unroll 4
                    for (int row = r0; row < nrows; row += 8) {
                        const int off0 = s_rowm[row];
                        const float v0 = t0p[(row - r0) * kPitch];
                        if (off0 >= 0) __stcs(dstb + off0, v0);
                        if (row + 4 < nrows) {
                            const int off1 = s_rowm[row + 4];
                            const float v1 = t1p[(row - r0) * kPitch];
                            if (off1 >= 0) __stcs(dstb + off1, v1);
                        }
                    }
                } else
#pragma unroll 4
                for (int row = threadIdx.x >> 4; row < nrows; row += kRunNT / 16) {
                    const int off = s_rowm[row];
                    if (off < 0) continue;
                    const int64_t o = map_base + off + n + c;
                    if (want_map)
                        __stcs(pr.out_maps + o,
                               tile[(size_t)row * kPitch + 4 * (gsel ^ ((row >> 1) & 3)) + w]);
                    if (want_flags)
                        pr.out_flags[o] =
                            (uint8_t)((ftile[row * kFPitch + gsel] >> (8 * w)) & 0xffu);
                }
            }
            __syncthreads();
        }
    }

    if (MARG) {
        Marg mg;
        marg_init(mg);
        if (rm.nv > 0) {
            mg.best = rm.best;
            mg.idx = rm.idx;
            mg.M = 0.5f * rm.best;
            mg.S = rm.sum * ex2_approx(rm.ref2 - rm.best * kHalfLog2e);
            mg.nvalid = rm.nv;
        }
        marg_block_reduce<kRunNT>(mg, s_red);
        if (threadIdx.x == 0) partial_store(partials + blockIdx.x, mg);
    }
}


// ---------------------------------------------------------------------------------------
// rect_tile_kernel: the rectangular map in its DIRECT form, tile by tile, for grids whose lattice
// steps are small (dt0 and dtau within a factor 4 of each other: the paper's full-resolution
// setups).
//
// Every cell is S(m, n) = P[hi(m, n)] - P[lo_m].  A CTA owns TR rows x TC columns and picks an
// anchor atom a at the low end of its window ENDS; in fp64 it stages, once,
//     Phi[j] = P[edge[j]] - P[a]   for the few hundred lattice points j the tile touches, and
//     U[m]   = P[a] - P[lo_m]      for its rows,
// rounded to fp32 (32 bytes each).  A cell is then Phi[j(m, n)] + U[m]: 8 additions, no running
// sum, no dependency between cells, no restart.  As long as the anchor lies inside the window
// (lo_m <= a <= hi) both terms are partial sums of the window and the fp32 rounding is that of
// the window's own sums; where it does not (short windows in the first column tile) the cell is
// sent to the fp64 path whenever the sum is smaller than an eighth of the larger term.
//
// The cells (m, n) and (m + r, n - c) with r e_m = c e_n sit on the SAME lattice point: a thread
// takes them as one packed pair -- Phi is a broadcast operand, U a row pair -- and closes them
// with the packed eq. (7) of pair_closure.  Lanes run along n, so both cells of a pair are stored
// by plain coalesced 128-byte warp stores: no shared-memory transpose, no barrier in the loop.
// Per cell: 16 bytes of shared-memory reads (the running-sum kernel: 32 + the transpose).
// ---------------------------------------------------------------------------------------
constexpr int kTileNT = 128;
constexpr int kTileNH = 1;                       // packed cell pairs per thread and lattice point
constexpr int kTileCells = 2 * kTileNH;          // cells per thread and lattice point
constexpr int kTileQuads = kTileNT / kTileCells;  // such groups of rows per CTA (128 rows)
constexpr int kTileCols = 256;  // columns per CTA
constexpr int kTileMaxRun = 768;  // lattice points a tile may touch (24 KB of shared memory)
constexpr float kTileSafeMag = 1073741824.0f;  // 2^30: below it eq. (7) cannot overflow in fp32
constexpr float kAnchorGuard = 8.0f;
constexpr int kTileGroup = 4 / kTileNH;  // column strips of a group summed as one straight-line block

// eq. (7) for two cells on the tile kernel's channels: 0 A, 1 B, 2 C/2, 3 -2C, 4..7 sqrt2 (Re Fa,
// Im Fa, Re Fb, Im Fb), so that D = A B + (-2C)(C/2) and the cross term is one multiply-add.
// SAFE: every staged value of the CTA is below 2^30 in magnitude, so nothing can overflow and
// the fast path holds where t = D - A B / 64 > kTiny (13 packed operations); otherwise t also
// carries the -kTiny offset and the overflow poison of pair_closure.
template <bool SAFE>
__device__ __forceinline__ PairOut pair_closure_tile(const u64 (&S)[8])
{
    const u64 p = fmul2(S[0], S[1]);
    u64 D = p;
    ffma2(D, S[3], S[2]);
    PairOut o;
    o.t = SAFE ? D : fadd2(D, pack2(-kTiny, -kTiny));
    ffma2(o.t, p, pack2(-kCondFast, -kCondFast));
    u64 na = fmul2(S[4], S[4]);
    ffma2(na, S[5], S[5]);
    u64 nb = fmul2(S[6], S[6]);
    ffma2(nb, S[7], S[7]);
    u64 re = fmul2(S[4], S[6]);
    ffma2(re, S[5], S[7]);
    u64 num = fmul2(S[1], na);
    ffma2(num, S[0], nb);
    ffma2(num, S[3], re);
    if (!SAFE) ffma2(o.t, fmul2(num, p), 0ull);
    float d0, d1;
    unpack2(D, d0, d1);
    o.res = fmul2(num, pack2(rcp_approx(d0), rcp_approx(d1)));
    return o;
}

// marginal update of one thread for two cells (values -inf where a cell does not count)
__device__ __forceinline__ void tile_marg2(RunMarg &rm, const float x0, const float x1,
                                           const int32_t flat0, const int32_t flat1)
{
    const float gmax = fmaxf(x0, x1);
    if (gmax >= rm.best && gmax > -INFINITY) {
        // rare: a new maximum, or an exact tie (the lowest flat index wins)
        int32_t cand = 0x7fffffff;
        if (x0 == gmax) cand = flat0;
        if (x1 == gmax) cand = min(cand, flat1);
        if (gmax > rm.best || cand < rm.idx) rm.idx = cand;
        rm.best = gmax;
    }
    if (fmaf(gmax, kHalfLog2e, -rm.ref2) > 60.0f) {  // rare: move the reference
        rm.sum *= ex2_approx(rm.ref2 - gmax * kHalfLog2e);
        rm.ref2 = gmax * kHalfLog2e;
    }
    rm.sum += ex2_approx(fmaf(x0, kHalfLog2e, -rm.ref2)) + ex2_approx(fmaf(x1, kHalfLog2e, -rm.ref2));
    rm.nv += (x0 > -INFINITY ? 1 : 0) + (x1 > -INFINITY ? 1 : 0);
}

// A thread's unit of work is a GROUP of kTileCells cells (m, n), (m + r, n - c), (m + 2r, n - 2c),
// .. which all sit on the lattice point j = m e_m + n e_n, as kTileNH packed pairs that share one
// Phi[j].  Measured on B200 (one-year map): one pair per thread 390 us (112 registers), two pairs
// 400 us (128 registers: half the shared-memory wavefronts, but fewer independent eq. (7) chains
// in flight and more address arithmetic per store).
// EN: the lattice step e_n of a column if it is 1 (the full-resolution grids: strides become
// immediates), 0 = taken from the bounds tables.
template <bool MARG, bool FLAGS, bool MAP, int EN>
__global__ void __launch_bounds__(kTileNT, 6)
    rect_tile_kernel(const Problem pr, const double *__restrict__ prefix,
                     Partial *__restrict__ partials, const int r, const int c, const int n_rowtiles,
                     const int n_coltiles)
{
    __shared__ __align__(16) float4 s_phiA[kTileMaxRun];  // A, B, C/2, -2C
    __shared__ __align__(16) float4 s_phiB[kTileMaxRun];  // sqrt2 (Re Fa, Im Fa, Re Fb, Im Fb)
    __shared__ __align__(16) u64 s_u[kTileQuads][kTileNH][8];  // channel pairs (U[m0], U[m1]), ..
    __shared__ int s_nfirst[kTileQuads][kTileCells];              // first column with >= min_atoms atoms
    __shared__ int s_row0[kTileQuads];                    // first row of quad q
    __shared__ unsigned s_mag;                            // largest staged magnitude (float bits)
    __shared__ Marg s_red[32];

    const Grid g = pr.grid;
    const Bounds &bd = pr.bounds;
    const int e_n = EN ? EN : bd.e_n;
    const int rowtile = blockIdx.x % n_rowtiles;
    const int coltile = (blockIdx.x / n_rowtiles) % n_coltiles;
    const int tpl = blockIdx.x / (n_rowtiles * n_coltiles);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int m0 = rowtile * (kTileCells * kTileQuads);
    const int n0 = coltile * kTileCols;
    const double2 *__restrict__ P =
        reinterpret_cast<const double2 *>(prefix + (int64_t)tpl * (bd.n_atoms + 1) * 8);

    // ---- staging ---------------------------------------------------------------------------
    // lattice points of the tile: those of the quads' first cells (m, n0 .. n0 + TC - 1)
    const int j_lo = (int)min((int64_t)m0 * bd.e_m + (int64_t)n0 * bd.e_n, (int64_t)bd.J - 1);
    const int j_hi = (int)min((int64_t)(m0 + kTileCells * kTileQuads - (kTileCells - 1) * r - 1) * bd.e_m +
                                  (int64_t)(n0 + kTileCols - 1) * bd.e_n,
                              (int64_t)bd.J - 1);
    const int a = __ldg(bd.edge + j_lo);  // the anchor: the smallest window end of the tile
    const double2 a0 = __ldg(P + (int64_t)a * 4), a1 = __ldg(P + (int64_t)a * 4 + 1),
                  a2 = __ldg(P + (int64_t)a * 4 + 2), a3 = __ldg(P + (int64_t)a * 4 + 3);
    // P[i] - P[a] as the 8 fp32 channels; NaN if a non-finite atom lies between the two
    auto rel = [&](const int i, float(&v)[8]) {
        const double2 h0 = __ldg(P + (int64_t)i * 4), h1 = __ldg(P + (int64_t)i * 4 + 1),
                      h2 = __ldg(P + (int64_t)i * 4 + 2), h3 = __ldg(P + (int64_t)i * 4 + 3);
        const double cc = h1.x - a1.x;
        v[0] = (float)(h0.x - a0.x);
        v[1] = (float)(h0.y - a0.y);
        v[2] = (float)(0.5 * cc);
        v[3] = (float)(-2.0 * cc);
        v[4] = (float)(kSqrt2 * (h1.y - a1.y));
        v[5] = (float)(kSqrt2 * (h2.x - a2.x));
        v[6] = (float)(kSqrt2 * (h2.y - a2.y));
        v[7] = (float)(kSqrt2 * (h3.x - a3.x));
        if (fabs(h3.y - a3.y) > 0.5) v[0] = nanf("");  // a bad SFT in between: fp64 path decides
    };
    if (threadIdx.x == 0) s_mag = 0u;
    unsigned mag_bits = 0u;  // (a NaN's bit pattern is above that of any finite value)
    auto track = [&](const float(&v)[8]) {
#pragma unroll
        for (int k = 0; k < 8; ++k) mag_bits = max(mag_bits, __float_as_uint(fabsf(v[k])));
    };
    static_assert(kTileCells * kTileQuads == kTileNT, "one thread per row of the tile");
    {
        // row of this thread: group q, member k4; U[m] = P[a] - P[lo_m]
        const int q = threadIdx.x / kTileCells, k4 = threadIdx.x % kTileCells;
        const int mq = m0 + (q / r) * kTileCells * r + q % r;
        const int m = mq + k4 * r;
        float v[8];
        int nfirst = 0x7fffffff;  // rows outside the map: no cell
        if (m < g.N_t0) {
            const int lo = __ldg(bd.lo + m);
            rel(lo, v);
            track(v);
            // first column of the row with at least min_atoms atoms (counts grow with n); mostly
            // the very first one: a search only where it is not
            int x = 0, e = g.N_tau;
            if (__ldg(bd.edge + (int64_t)m * bd.e_m) - lo >= pr.min_atoms) e = 0;
            while (x < e) {
                const int mid = (x + e) >> 1;
                const int cnt = __ldg(bd.edge + (int64_t)m * bd.e_m + (int64_t)mid * bd.e_n) - lo;
                if (cnt < pr.min_atoms) x = mid + 1;
                else e = mid;
            }
            nfirst = x;
        } else {
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = 0.0f;
            v[0] = v[1] = -1.0e15f;  // a dummy, perfectly conditioned row
        }
        float *u = reinterpret_cast<float *>(&s_u[q][k4 >> 1][0]);
#pragma unroll
        for (int k = 0; k < 8; ++k) u[2 * k + (k4 & 1)] = -v[k];
        s_nfirst[q][k4] = nfirst;
        if (k4 == 0) s_row0[q] = mq;
    }
    for (int jj = threadIdx.x; jj <= j_hi - j_lo; jj += kTileNT) {
        float v[8];
        rel(__ldg(bd.edge + j_lo + jj), v);
        track(v);
        s_phiA[jj] = make_float4(v[0], v[1], v[2], v[3]);
        s_phiB[jj] = make_float4(v[4], v[5], v[6], v[7]);
    }
    mag_bits = __reduce_max_sync(0xffffffffu, mag_bits);
    __syncthreads();  // s_mag = 0 is in place
    if (lane == 0) atomicMax(&s_mag, mag_bits);
    __syncthreads();
    const bool mag_ok = s_mag <= __float_as_uint(kTileSafeMag);

    // ---- cells -------------------------------------------------------------------------------
    RunMarg rm;
    rm.best = -INFINITY;
    rm.idx = 0x7fffffff;
    rm.ref2 = -1.0e30f;
    rm.sum = 0.0f;
    rm.nv = 0;
    const int64_t map_base = (int64_t)tpl * g.N_t0 * g.N_tau;
    float *__restrict__ const maps = MAP ? pr.out_maps + map_base : nullptr;
    uint8_t *__restrict__ const flg = FLAGS ? pr.out_flags + map_base : nullptr;
    constexpr int n_strips = kTileCols / 32;
    // every cell of the tile lies inside the map
    const bool interior =
        m0 + kTileCells * kTileQuads <= g.N_t0 && n0 - (kTileCells - 1) * c >= 0 &&
        n0 + kTileCols <= g.N_tau;
    // a warp takes quads warp, warp + 4, ..: U and the row addresses stay in registers while it
    // walks the quad's column strips
#pragma unroll 1
    for (int q = warp; q < kTileQuads; q += kTileNT / 32) {
        const int mq = s_row0[q];
        if (mq >= g.N_t0) continue;
        u64 U[kTileNH][8];
#pragma unroll
        for (int h = 0; h < kTileNH; ++h)
#pragma unroll
            for (int k = 0; k < 8; ++k) U[h][k] = s_u[q][h][k];
        float ua[kTileCells];
#pragma unroll
        for (int h = 0; h < kTileNH; ++h) unpack2(U[h][0], ua[2 * h], ua[2 * h + 1]);
        int nf[kTileCells];
#pragma unroll
        for (int k = 0; k < kTileCells; ++k) nf[k] = s_nfirst[q][k];
        const int jl = (int)((int64_t)mq * bd.e_m + (int64_t)n0 * bd.e_n - j_lo) + lane * bd.e_n;
        int32_t flat0[kTileCells];  // flat index of the group's cells at strip 0
#pragma unroll
        for (int k = 0; k < kTileCells; ++k) flat0[k] = (mq + k * r) * g.N_tau + n0 - k * c + lane;
        // lean: interior tile, values in range, the anchor inside every window of the quad
        // (U >= 0: lo_m <= a), and enough atoms from the tile's first column on
        bool lean = interior && mag_ok;
#pragma unroll
        for (int k = 0; k < kTileCells; ++k) lean = lean && ua[k] >= 0.0f && nf[k] <= n0 - k * c;
        if (lean) {
            // kTileGroup strips of the quad as ONE straight-line block: their eq. (7) chains are
            // independent and interleave (a branch per strip would fence them off from one
            // another); the rare cells that fail the conditioning test are redone afterwards.
            // Addresses are carried as pointers that advance by one block per trip, so that a
            // strip's loads and stores take immediate offsets (ncu before: 59 of the 170
            // instructions of a block were address arithmetic and the conditioning test).
            const int jstep = 32 * e_n;  // lattice points per strip
            const float4 *pA = s_phiA + jl, *pB = s_phiB + jl;
            float *pm[kTileCells];
            uint8_t *pf[kTileCells];
#pragma unroll
            for (int k = 0; k < kTileCells; ++k) {
                pm[k] = MAP ? maps + flat0[k] : nullptr;
                pf[k] = FLAGS ? flg + flat0[k] : nullptr;
            }
#pragma unroll 1
            for (int s0 = 0; s0 < n_strips; s0 += kTileGroup) {
                float res[kTileGroup][kTileCells];
                u64 tt2[kTileGroup][kTileNH];
#pragma unroll
                for (int strip = 0; strip < kTileGroup; ++strip) {
                    const float4 fa = pA[strip * jstep], fb = pB[strip * jstep];
                    const u64 ph[8] = {pack2(fa.x, fa.x), pack2(fa.y, fa.y), pack2(fa.z, fa.z),
                                       pack2(fa.w, fa.w), pack2(fb.x, fb.x), pack2(fb.y, fb.y),
                                       pack2(fb.z, fb.z), pack2(fb.w, fb.w)};
#pragma unroll
                    for (int h = 0; h < kTileNH; ++h) {
                        u64 S[8];
#pragma unroll
                        for (int k = 0; k < 8; ++k) S[k] = fadd2(ph[k], U[h][k]);
                        const PairOut o = pair_closure_tile<true>(S);
                        unpack2(o.res, res[strip][2 * h], res[strip][2 * h + 1]);
                        tt2[strip][h] = o.t;
                    }
                }
                // one test for the whole block (fminf drops a NaN, so NaNs are looked for with
                // the sum, taken pairwise); which cells failed is only worked out in the rare case
                // that one did
                float tt[kTileGroup][kTileCells];
                u64 ts2 = tt2[0][0];
#pragma unroll
                for (int strip = 0; strip < kTileGroup; ++strip)
#pragma unroll
                    for (int h = 0; h < kTileNH; ++h) {
                        unpack2(tt2[strip][h], tt[strip][2 * h], tt[strip][2 * h + 1]);
                        if (strip + h) ts2 = fadd2(ts2, tt2[strip][h]);
                    }
                float tmin = tt[0][0], ts_lo, ts_hi;
#pragma unroll
                for (int strip = 0; strip < kTileGroup; ++strip)
#pragma unroll
                    for (int k = 0; k < kTileCells; ++k) tmin = fminf(tmin, tt[strip][k]);
                unpack2(ts2, ts_lo, ts_hi);
                const float tsum = ts_lo + ts_hi;
                uint32_t fl = 0u;  // D <= 0 / count flags of the redone cells, 2 bits per cell
                if (!(tmin > kTiny) || !(tsum == tsum)) {  // rare: the plain way, in fp64 from P
                    const int jg = (int)(pA - s_phiA);
                    uint32_t slow = 0u;
#pragma unroll
                    for (int strip = 0; strip < kTileGroup; ++strip)
#pragma unroll
                        for (int k = 0; k < kTileCells; ++k)
                            slow |= (tt[strip][k] > kTiny ? 0u : 1u) << (kTileCells * strip + k);
#pragma unroll
                    for (int strip = 0; strip < kTileGroup; ++strip) {
                        const int64_t j = (int64_t)j_lo + jg + strip * jstep;
#pragma unroll
                        for (int k = 0; k < kTileCells; ++k) {
                            if (slow & (1u << (kTileCells * strip + k))) {
                                float flf;
                                unpack2(rect_cell_slow(P, bd.lo, bd.edge, mq + k * r, j,
                                                       pr.min_atoms),
                                        res[strip][k], flf);
                                fl |= (__float_as_uint(flf) & 3u) << (2 * (kTileCells * strip + k));
                            }
                        }
                    }
                }
#pragma unroll
                for (int strip = 0; strip < kTileGroup; ++strip) {
                    float x[kTileCells];
#pragma unroll
                    for (int k = 0; k < kTileCells; ++k) {
                        const uint32_t f = (fl >> (2 * (kTileCells * strip + k))) & 3u;
                        if (MAP) __stcs(pm[k] + 32 * strip, res[strip][k]);
                        if (FLAGS) pf[k][32 * strip] = (uint8_t)f;
                        x[k] = f ? -INFINITY : res[strip][k];
                    }
                    if (MARG) {
#pragma unroll
                        for (int h = 0; h < kTileNH; ++h)
                            tile_marg2(rm, x[2 * h], x[2 * h + 1], flat0[2 * h] + 32 * (s0 + strip),
                                       flat0[2 * h + 1] + 32 * (s0 + strip));
                    }
                }
                pA += kTileGroup * jstep;
                pB += kTileGroup * jstep;
#pragma unroll
                for (int k = 0; k < kTileCells; ++k) {
                    if (MAP) pm[k] += 32 * kTileGroup;
                    if (FLAGS) pf[k] += 32 * kTileGroup;
                }
            }
        } else {
            // edge tiles, short windows, values far from unity: every cell is tested for being
            // inside the map, for its atom count and for an anchor outside its window
#pragma unroll 1
            for (int strip = 0; strip < n_strips; ++strip) {
                const int n = n0 + 32 * strip + lane;
                if (n0 + 32 * strip - (kTileCells - 1) * c >= g.N_tau) break;  // beyond the map
                const int jj = min(jl + 32 * strip * bd.e_n, j_hi - j_lo);
                const int64_t j = (int64_t)mq * bd.e_m + (int64_t)n * bd.e_n;
                const float4 fa = s_phiA[jj], fb = s_phiB[jj];
                const u64 ph[8] = {pack2(fa.x, fa.x), pack2(fa.y, fa.y), pack2(fa.z, fa.z),
                                   pack2(fa.w, fa.w), pack2(fb.x, fb.x), pack2(fb.y, fb.y),
                                   pack2(fb.z, fb.z), pack2(fb.w, fb.w)};
                float x[kTileCells];
#pragma unroll
                for (int h = 0; h < kTileNH; ++h) {
                    u64 S[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) S[k] = fadd2(ph[k], U[h][k]);
                    const PairOut o = pair_closure_tile<false>(S);
                    float rr[2], tt[2], sa[2];
                    unpack2(o.res, rr[0], rr[1]);
                    unpack2(o.t, tt[0], tt[1]);
                    unpack2(S[0], sa[0], sa[1]);
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int k = 2 * h + e;
                        const int m = mq + k * r, nk = n - k * c;
                        const bool ok = m < g.N_t0 && nk >= 0 && nk < g.N_tau;
                        // an anchor outside the window: the sum must not be a small difference
                        // of the two terms
                        const bool fast = tt[e] > 0.0f && nk >= nf[k] &&
                                          sa[e] * kAnchorGuard >= fmaxf(fabsf(fa.x), fabsf(ua[k]));
                        uint32_t f = 0u;
                        if (ok && !fast) {  // the plain way, in fp64 from P
                            float flf;
                            unpack2(rect_cell_slow(P, bd.lo, bd.edge, m, j, pr.min_atoms), rr[e],
                                    flf);
                            f = __float_as_uint(flf);
                        }
                        const int32_t flat = flat0[k] + 32 * strip;
                        if (ok) {
                            if (MAP) __stcs(maps + flat, rr[e]);
                            if (FLAGS) flg[flat] = (uint8_t)f;
                        }
                        x[k] = (ok && f == 0u) ? rr[e] : -INFINITY;
                    }
                }
                if (MARG) {
#pragma unroll
                    for (int h = 0; h < kTileNH; ++h)
                        tile_marg2(rm, x[2 * h], x[2 * h + 1], flat0[2 * h] + 32 * strip,
                                   flat0[2 * h + 1] + 32 * strip);
                }
            }
        }
    }
    if (MARG) {
        Marg mg;
        marg_init(mg);
        if (rm.nv > 0) {
            mg.best = rm.best;
            mg.idx = rm.idx;
            mg.M = 0.5f * rm.best;
            mg.S = rm.sum * ex2_approx(rm.ref2 - rm.best * kHalfLog2e);
            mg.nvalid = rm.nv;
        }
        marg_block_reduce<kTileNT>(mg, s_red);
        if (threadIdx.x == 0) partial_store(partials + blockIdx.x, mg);
    }
}

cudaError_t launch_tile(const Plan &pl, const Problem &pr, const double *prefix, Partial *partials,
                        cudaStream_t st)
{
    const RectRun &rr = pl.rect;
    const int64_t n_ctas = (int64_t)rr.n_rowtiles * rr.n_coltiles * pl.n_templates;
    auto go = [&](auto kern) {
        return launch_k(kern, (unsigned)n_ctas, kTileNT, 0, st, pr, prefix, partials, rr.r, rr.NTu,
                          rr.n_rowtiles, rr.n_coltiles);
    };
    const bool e1 = pl.e_n == 1;
#define TFSTAT_TILE_GO(M, F, P) \
    (e1 ? go(rect_tile_kernel<M, F, P, 1>) : go(rect_tile_kernel<M, F, P, 0>))
    if (pr.out_flags) {
        if (pr.out_maps)
            return partials ? TFSTAT_TILE_GO(true, true, true) : TFSTAT_TILE_GO(false, true, true);
        return partials ? TFSTAT_TILE_GO(true, true, false) : TFSTAT_TILE_GO(false, true, false);
    }
    if (pr.out_maps)
        return partials ? TFSTAT_TILE_GO(true, false, true) : TFSTAT_TILE_GO(false, false, true);
    return TFSTAT_TILE_GO(true, false, false);
#undef TFSTAT_TILE_GO
}

template <int Q>
cudaError_t launch_run(const Plan &pl, const Problem &pr, const double *prefix,
                       const ulonglong2 *K, Partial *partials, cudaStream_t st)
{
    const RectRun &rr = pl.rect;
    const int nrows = Q * kRunNT;
    // the flag tile is only there when flags are asked for: shared memory not taken is L1
    const size_t smem = (size_t)nrows * (kPitch * 4 + 4 + (pr.out_flags ? kFPitch * 4 : 0));
    const int64_t cells = (int64_t)pl.grid.N_t0 * pl.grid.N_tau;
    const bool vec = (pl.grid.N_tau % 4 == 0) && (cells % 4 == 0) &&
                     ((reinterpret_cast<uintptr_t>(pr.out_maps) & 15u) == 0) &&
                     ((reinterpret_cast<uintptr_t>(pr.out_flags) & 3u) == 0);
    const int64_t n_ctas = (int64_t)rr.n_rowtiles * rr.n_coltiles * pl.n_templates;
    const int ks_cap = rr.ks_cap;
    const bool ks = ks_cap > 0;
    const size_t smem_all = smem + (size_t)ks_cap * 64;
    auto go = [&](auto kern) -> cudaError_t {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)smem_all);
        if (e != cudaSuccess) return e;
        return launch_k(kern, (unsigned)n_ctas, kRunNT, smem_all, st, pr, prefix, K, partials,
                          rr.r, rr.NTu, rr.seg_cols, rr.n_rowtiles, rr.n_coltiles, vec ? 1 : 0,
                          ks_cap, rr.ks_lg);
    };
    if (partials) return ks ? go(rect_run_kernel<Q, true, true>) : go(rect_run_kernel<Q, true, false>);
    return ks ? go(rect_run_kernel<Q, false, true>) : go(rect_run_kernel<Q, false, false>);
}

}  // namespace

// Tile shapes of the running-sum kernel; called by make_plan (api.cu).
RectRun plan_rect_run(const Grid &g, int32_t e_m, int32_t e_n, int64_t J, int32_t n_templates,
                      int32_t q_override, int32_t seg_override)
{
    RectRun rr;
    rr.enabled = (J > 0 && g.N_t0 >= 8) ? 1 : 0;
    rr.tile = 0;
    // direct form, tile by tile (rect_tile_kernel): lattice steps small enough for a tile's run of
    // lattice points to sit in shared memory; seg_override < 0 keeps the running-sum kernel
    // (q_override == 8 forces it on any grid whose lattice qualifies: the tests' small maps)
    if (rr.enabled && e_m >= 1 && e_n >= 1 && e_m <= 4 && e_n <= 4 && seg_override >= 0 &&
        (q_override == 0 || q_override == 8) && (kTileQuads % e_n) == 0 &&
        (int64_t)(kTileCells * kTileQuads - (kTileCells - 1) * e_n - 1) * e_m +
                (int64_t)(kTileCols - 1) * e_n + 1 <=
            kTileMaxRun) {
        const int64_t n_rt = (g.N_t0 + kTileCells * kTileQuads - 1) / (kTileCells * kTileQuads);
        const int64_t n_ct = (g.N_tau + (kTileCells - 1) * e_m + kTileCols - 1) / kTileCols;
        // (a small map gives too few 128 x 256 tiles to fill 148 SMs: config 3's 96 x 5736 cells
        // are 23 tiles, 58 us against 44 us for the running-sum kernel)
        if (n_rt * n_ct * n_templates >= 2 * 148 || q_override == 8) rr.tile = 1;
    }
    if (rr.tile) {
        rr.Q = kTileCells;
        rr.r = e_n;    // rows m, m + r, ...
        rr.NTu = e_m;  // ... meet on one lattice point, c = e_m columns apart each
        rr.seg_cols = kTileCols;
        rr.n_rowtiles = (g.N_t0 + kTileCells * kTileQuads - 1) / (kTileCells * kTileQuads);
        rr.n_coltiles = (g.N_tau + (kTileCells - 1) * e_m + kTileCols - 1) / kTileCols;
        rr.ks_cap = 0;
        rr.ks_lg = -1;
        return rr;
    }
    rr.Q = 1;
    rr.r = 1;
    bool perm_ok = false;
    // Row m + roff, roff = 2 e_n / e_m, sits at column n on the lattice point that row m
    // reaches two columns (one pair-step) later: a thread that owns both loads every K entry
    // once for two rows.
    if (e_m > 0 && e_n > 0 && (2 * (int64_t)e_n) % e_m == 0 && q_override != 1) {
        const int64_t roff = 2 * (int64_t)e_n / e_m;
        // ... if a warp still reads K in runs of 16 lattice points (roff >= 16).  For dt0 = dtau
        // (roff = 2) the lanes of a row pair touch every other pair of entries, and one row per
        // thread is faster although it loads K twice -- also when the run is staged in shared
        // memory in two conflict-free halves (ks_lg, used when two rows are forced for dtau =
        // dt0 or 2 dt0): one-year map at full resolution 646 us against 561 us.
        perm_ok = e_m == 1 && (roff == 2 || roff == 4);
        const bool two = roff >= 16 || q_override == 2;
        if (g.N_t0 >= 2 * roff && two) {
            rr.Q = 2;
            rr.r = (int32_t)roff;
        }
    }
    // NTu = R: residues per CTA (a power of two <= 16, so that a warp still reads K in runs of
    // at least min(roff, 16) x 16 bytes); the CTA's other lanes hold the following groups
    int R = 16;
    while (R > rr.r) R >>= 1;
    rr.NTu = rr.Q > 1 ? R : kRunNT;
    if (rr.Q > 1) {
        const int64_t groups = ((int64_t)g.N_t0 + (int64_t)rr.r * rr.Q - 1) / ((int64_t)rr.r * rr.Q);
        const int64_t gpc = kRunNT / R;
        rr.n_rowtiles = (int32_t)(((rr.r + R - 1) / R) * ((groups + gpc - 1) / gpc));
    } else {
        rr.n_rowtiles = (int32_t)(((int64_t)g.N_t0 + kRunNT - 1) / kRunNT);
    }
    // columns per CTA: whole waves of 148 SMs x resident CTAs; a row start costs about as
    // much as 24 cells
    const int seg_max = (g.N_tau + kChunk - 1) / kChunk * kChunk;
    int seg = seg_max;
    int64_t best_cost = INT64_MAX;
    // lattice points one CTA walks: its rows' starting points plus the pair-steps of one row
    // (the loads run NS ahead of their use; what lies beyond the run is never used)
    auto ks_span = [&](const int sc) -> int64_t {
        const int64_t row_span =
            rr.Q == 1 ? kRunNT - 1 : (int64_t)(kRunNT / R - 1) * rr.r * rr.Q + R - 1;
        return row_span * e_m + (int64_t)(2 * ((sc + 3) / 4) + rr.Q) * 2 * e_n + 1;
    };
    // plenty of CTAs even with short column tiles: the widest of 192, 128, 64 columns whose K
    // run still fits in shared memory (one-year map at full resolution, K staged: 64 columns
    // 646 us, 128 586 us, 192 570 us, 256 -- K from L1 again -- 657 us; short fp32 running sums
    // besides)
    // 8 CTAs per SM: 64-byte entries beside the transposed tile (4 KB, two rows per thread 8 KB)
    const int ks_max = rr.Q == 1 ? kKsMaxEntries : kKsMaxEntries - 32;
    bool plenty = false;
    for (const int pref : {192, 128, 64}) {
        const int sp = std::min(seg_max, pref);
        if ((int64_t)n_templates * rr.n_rowtiles * ((g.N_tau + sp - 1) / sp) < (int64_t)148 * 8 * 16)
            continue;
        if (pref > 64 && ks_span(sp) > ks_max) continue;
        plenty = true;
        seg = sp;
        break;
    }
    for (int cand = seg_max; !plenty && cand >= kChunk; cand -= kChunk) {
        const int64_t ctas = (int64_t)n_templates * rr.n_rowtiles * ((g.N_tau + cand - 1) / cand);
        const int64_t per_wave = 148 * 8;
        const int64_t waves = (ctas + per_wave - 1) / per_wave;
        const int64_t cost = waves * (cand + 24);
        if (cost < best_cost) {
            best_cost = cost;
            seg = cand;
        }
        if (ctas >= (int64_t)148 * 4 * 64) break;  // many waves: quantisation no longer matters
    }
    if (seg_override > 0) seg = std::min(seg_max, (seg_override + kChunk - 1) / kChunk * kChunk);
    rr.seg_cols = seg;
    rr.n_coltiles = (g.N_tau + seg - 1) / seg;
    rr.ks_cap = ks_span(seg) <= ks_max ? (int32_t)ks_span(seg) : 0;
    rr.ks_lg = -1;
    if (rr.ks_cap > 0 && rr.Q == 2 && perm_ok && R == rr.r) {
        rr.ks_lg = R == 2 ? 1 : 2;
        rr.ks_cap = 2 * R * ((rr.ks_cap - 1) / (2 * R) + 1);  // two halves, whole runs of R
    }
    return rr;
}

// One CTA per template pays off while the map is small, or while the templates alone fill the GPU
bool rect_small_applies(int32_t n_atoms, int32_t n_templates, int64_t cells)
{
    if (n_atoms > 2048) return false;  // 64 B of fp64 prefix + 4 B per atom in shared memory
    return cells <= 4096 || (n_templates >= 148 * 4 && cells <= 32768);
}

cudaError_t launch_rect_small(const Plan &pl, const Problem &pr, cudaStream_t st)
{
    const size_t smem = (size_t)(pl.n_atoms + 1) * 64 + (size_t)pl.n_atoms * 5;
    cudaError_t e = cudaFuncSetAttribute(rect_small_kernel,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    rect_small_kernel<<<(unsigned)pl.n_templates, kSmallNT, smem, st>>>(pr);
    return cudaGetLastError();
}

int rect_run_threads(const Plan &pl) { return pl.rect.tile ? kTileNT : kRunNT; }

int rect_scan_blocks(int32_t n_atoms) { return (n_atoms + kScanBlock - 1) / kScanBlock; }

cudaError_t launch_rect(const Plan &pl, const Problem &pr, double *prefix, double *agg,
                        int32_t *flags, void *steps, Partial *partials, cudaStream_t st)
{
    // flags (ready + done per scan block) must be zero here: launch_bounds zeroes them, and
    // run_device memsets them when the bounds of an earlier call are reused
    const int nblk = rect_scan_blocks(pl.n_atoms);
    const int n_scan = nblk * pl.n_templates;
    ulonglong2 *K = static_cast<ulonglong2 *>(steps);
    // (the tile kernel works from P alone: no step table)
    const int spt = pl.rect.enabled && !pl.rect.tile ? (int)((pl.J + 1 + kStepPts - 1) / kStepPts) : 0;
    const int64_t n_blocks = (int64_t)n_scan + (int64_t)spt * pl.n_templates;
    cudaError_t e = launch_k(rect_scan_kernel, (unsigned)n_blocks, kScanNT, 0, st, pr, agg, flags,
                               prefix, K, nblk, n_scan, spt);
    if (e != cudaSuccess) return e;
    if (!pl.rect.enabled) {
        const int64_t n_ctas = (int64_t)pl.cell_blocks_per_template * pl.n_templates;
        return launch_k(rect_cells_kernel, (unsigned)n_ctas, kCellNT, 0, st, pr, prefix, partials,
                          pl.cell_blocks_per_template);
    }
    if (pl.rect.tile) return launch_tile(pl, pr, prefix, partials, st);
    if (pl.rect.Q == 2) return launch_run<2>(pl, pr, prefix, K, partials, st);
    return launch_run<1>(pl, pr, prefix, K, partials, st);
}

}  // namespace tfstat
