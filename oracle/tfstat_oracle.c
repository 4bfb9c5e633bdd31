/*
 * tfstat_oracle.c -- fp64 CPU ORACLE for the transient F-statistic map.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant with the CUDA path under
 * paper_1805_05652_b200/ and must never be imported from there.
 *
 * It is the paper's definitions written out, cell by cell, with no blocking, prefix
 * sums, fusion or reordering:
 *
 *   window membership  PAPER.md:41-48, eqs. (3),(4): rectangular [t0, t0+tau),
 *                      exponential [t0, t0+3 tau) -- HALF-OPEN on atom start times,
 *                      the reading fixed by the paper's own term counts
 *                      (A.5)/(A.6), and "3 tau / T_SFT atoms",
 *                      PAPER.md:238.  Decided in integer seconds.
 *   weights            rect: 1;  exp: w = exp(-(t - t0)/tau), libm fp64
 *                      (eq. 4; libm exp as in the paper's accuracy
 *                      check).
 *   where w enters     linear on Fa, Fb; quadratic on a2, b2, ab
 *                      (h = varpi * h_CW, and eq. (6)).
 *   truncation         only existing atoms contribute; windows overrunning the data
 *                      (or starting before it, or spanning gaps) are simply shorter
 *                      sums and the full matrix is still returned.
 *   closure            D = A B - C^2 and eq. (7); the map
 *                      stores 2F.
 *   degenerate cells   fewer than `min_atoms` atoms (default 2: "at least 2 SFTs per
 *                      F_mn") -> flag bit 0;  !(D > 0) -> flag bit 1.
 *                      Degenerate cells store 2F = 0 and are excluded from the
 *                      marginals.  Atoms that are not finite are NOT special here:
 *                      the arithmetic is followed (a NaN in a2 / b2 / ab makes D NaN
 *                      -> bit 1; a NaN confined to Fa / Fb gives a NaN 2F with flag
 *                      0).  The paper is silent on bad SFTs: PARITY UNPINNED BY THE
 *                      PAPER; the GPU's convention is DESIGN.md reading R19.
 *   map layout         map[m*N_tau + n], m <-> t0, n <-> tau (eq. 8).
 *   marginals          max 2F over valid cells, lowest flat index on exact ties;
 *                      logB = log sum_valid exp(F), F = 2F/2 (eq. 5, PAPER.md:56;
 *                      c_marg footnote PAPER.md:227).  The paper does not print a
 *                      normalisation for logB: PARITY UNPINNED BY THE PAPER for the
 *                      constant offset; the convention is DESIGN.md reading R13.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute force by an independent
 * dense-weight-matrix formulation, the toy example tests/golden/T0_*.txt, the
 * closed form for injections (I1), full-span rect == CW F-statistic (I2), scale /
 * shift invariances (I3-I5), the integer term counts of (A.5)/(A.6) (I6), tau->inf
 * limit (I7), chi^2_4 noise statistics (I9).
 *
 * Inputs are fp32 (the paper's real32 atoms) promoted exactly to fp64.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_RECT 0
#define ORACLE_EXP 1

typedef struct {
    double max2F; /* 0 if n_valid == 0 */
    int32_t m, n; /* argmax, (-1,-1) if n_valid == 0 */
    double logB;  /* -inf if n_valid == 0 */
    int32_t n_valid;
    int32_t pad_;
} oracle_result;

typedef struct {
    double twoF;
    double cond;   /* D / (A B), oracle-only conditioning number (0 if A B == 0) */
    int32_t cnt;   /* atoms in the window */
    uint8_t flags; /* bit0: cnt < min_atoms, bit1: !(D > 0) */
} oracle_cell_t;

/* One grid cell by the literal definition.  atoms = 7 rows of stride ld:
 * a2, b2, ab, Re Fa, Im Fa, Re Fb, Im Fb. */
static oracle_cell_t oracle_cell(const float *atoms, int64_t ld, const int32_t *t,
                                 int32_t n_atoms, int window, int64_t t0, int64_t tau,
                                 int32_t min_atoms)
{
    const float *a2 = atoms, *b2 = atoms + ld, *ab = atoms + 2 * ld;
    const float *fare = atoms + 3 * ld, *faim = atoms + 4 * ld;
    const float *fbre = atoms + 5 * ld, *fbim = atoms + 6 * ld;
    const int64_t k = (window == ORACLE_EXP) ? 3 : 1;
    const int64_t t_end = t0 + k * tau;
    double A = 0, B = 0, C = 0, FaRe = 0, FaIm = 0, FbRe = 0, FbIm = 0;
    int32_t cnt = 0;
    for (int32_t al = 0; al < n_atoms; ++al) {
        const int64_t ta = t[al];
        if (ta < t0) continue;
        if (ta >= t_end) break; /* timestamps strictly increasing: nothing further */
        double w = 1.0;
        if (window == ORACLE_EXP) w = exp(-(double)(ta - t0) / (double)tau);
        const double w2 = w * w;
        A += w2 * (double)a2[al];
        B += w2 * (double)b2[al];
        C += w2 * (double)ab[al];
        FaRe += w * (double)fare[al];
        FaIm += w * (double)faim[al];
        FbRe += w * (double)fbre[al];
        FbIm += w * (double)fbim[al];
        cnt += 1;
    }
    oracle_cell_t r;
    const double D = A * B - C * C;
    r.cnt = cnt;
    r.flags = 0;
    if (cnt < min_atoms) r.flags |= 1;
    if (!(D > 0.0)) r.flags |= 2;
    r.cond = (A * B != 0.0) ? D / (A * B) : 0.0;
    if (r.flags) {
        r.twoF = 0.0;
    } else {
        const double F = (B * (FaRe * FaRe + FaIm * FaIm) + A * (FbRe * FbRe + FbIm * FbIm)
                          - 2.0 * C * (FaRe * FbRe + FaIm * FbIm)) / D; /* eq. (7) */
        r.twoF = 2.0 * F;
    }
    return r;
}

static int bad_args(const float *atoms, int64_t ld, const int32_t *t, int32_t n_atoms,
                    int window, int32_t N_t0, int32_t N_tau, int32_t tau_min)
{
    return !atoms || !t || n_atoms < 1 || ld < n_atoms || N_t0 < 1 || N_tau < 1 ||
           tau_min < 1 || (window != ORACLE_RECT && window != ORACLE_EXP);
}

/* Full map, eq. (8).  Any of out_flags/out_cond/out_cnt may be NULL. */
int oracle_tfstat_map(const float *atoms, int64_t ld, const int32_t *t, int32_t n_atoms,
                      int window, int32_t t0_min, int32_t dt0, int32_t N_t0,
                      int32_t tau_min, int32_t dtau, int32_t N_tau, int32_t min_atoms,
                      double *out_2F, uint8_t *out_flags, double *out_cond,
                      int32_t *out_cnt, int n_threads)
{
    if (bad_args(atoms, ld, t, n_atoms, window, N_t0, N_tau, tau_min) || !out_2F) return -1;
#ifdef _OPENMP
    if (n_threads < 1) n_threads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
#endif
    for (int32_t m = 0; m < N_t0; ++m) {
        for (int32_t n = 0; n < N_tau; ++n) {
            const int64_t t0 = (int64_t)t0_min + (int64_t)m * dt0;
            const int64_t tau = (int64_t)tau_min + (int64_t)n * dtau;
            const oracle_cell_t c =
                oracle_cell(atoms, ld, t, n_atoms, window, t0, tau, min_atoms);
            const int64_t i = (int64_t)m * N_tau + n;
            out_2F[i] = c.twoF;
            if (out_flags) out_flags[i] = c.flags;
            if (out_cond) out_cond[i] = c.cond;
            if (out_cnt) out_cnt[i] = c.cnt;
        }
    }
    return 0;
}

/* The same cell function on a list of K cells (ms[i], ns[i]) -- for sampled parity
 * at sizes where the full map would take too long. */
int oracle_tfstat_cells(const float *atoms, int64_t ld, const int32_t *t, int32_t n_atoms,
                        int window, int32_t t0_min, int32_t dt0, int32_t N_t0,
                        int32_t tau_min, int32_t dtau, int32_t N_tau, int32_t min_atoms,
                        const int32_t *ms, const int32_t *ns, int64_t K, double *out_2F,
                        uint8_t *out_flags, double *out_cond, int32_t *out_cnt,
                        int n_threads)
{
    if (bad_args(atoms, ld, t, n_atoms, window, N_t0, N_tau, tau_min) || !out_2F || !ms ||
        !ns)
        return -1;
#ifdef _OPENMP
    if (n_threads < 1) n_threads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 16) num_threads(n_threads)
#endif
    for (int64_t i = 0; i < K; ++i) {
        const int64_t t0 = (int64_t)t0_min + (int64_t)ms[i] * dt0;
        const int64_t tau = (int64_t)tau_min + (int64_t)ns[i] * dtau;
        const oracle_cell_t c = oracle_cell(atoms, ld, t, n_atoms, window, t0, tau, min_atoms);
        out_2F[i] = c.twoF;
        if (out_flags) out_flags[i] = c.flags;
        if (out_cond) out_cond[i] = c.cond;
        if (out_cnt) out_cnt[i] = c.cnt;
    }
    return 0;
}

/* Marginalise a map: max 2F (lowest flat index on ties) and logB = log sum exp(2F/2)
 * over cells with flags == 0 (flags NULL: every cell valid). */
int oracle_tfstat_marginalise(const double *map2F, const uint8_t *flags, int32_t N_t0,
                              int32_t N_tau, oracle_result *out)
{
    if (!map2F || !out || N_t0 < 1 || N_tau < 1) return -1;
    const int64_t n_cells = (int64_t)N_t0 * N_tau;
    double best = 0.0;
    int64_t arg = -1;
    int32_t n_valid = 0;
    for (int64_t i = 0; i < n_cells; ++i) {
        if (flags && flags[i]) continue;
        if (arg < 0 || map2F[i] > best) {
            best = map2F[i];
            arg = i;
        }
        n_valid += 1;
    }
    out->n_valid = n_valid;
    out->pad_ = 0;
    if (n_valid == 0) {
        out->max2F = 0.0;
        out->m = -1;
        out->n = -1;
        out->logB = -INFINITY;
        return 0;
    }
    double s = 0.0;
    for (int64_t i = 0; i < n_cells; ++i) {
        if (flags && flags[i]) continue;
        s += exp(0.5 * map2F[i] - 0.5 * best);
    }
    out->max2F = best;
    out->m = (int32_t)(arg / N_tau);
    out->n = (int32_t)(arg % N_tau);
    out->logB = 0.5 * best + log(s);
    return 0;
}

/* Batched search: T independent atom sets sharing timestamps and grid; per template the
 * full map by the definition, then its marginals (the paper's
 * per-template loop).  out_terms (nullable) receives the number of (cell, atom) terms
 * summed, the unit of work of eq. (A.6). */
int oracle_tfstat_search(const float *atoms, int64_t template_stride, int64_t ld,
                         const int32_t *t, int32_t n_atoms, int32_t n_templates, int window,
                         int32_t t0_min, int32_t dt0, int32_t N_t0, int32_t tau_min,
                         int32_t dtau, int32_t N_tau, int32_t min_atoms, oracle_result *out,
                         int64_t *out_terms, int n_threads)
{
    if (!atoms || n_templates < 1 || !out) return -1;
    if (bad_args(atoms, ld, t, n_atoms, window, N_t0, N_tau, tau_min)) return -1;
    const int64_t n_cells = (int64_t)N_t0 * N_tau;
    int rc = 0;
    int64_t terms = 0;
#ifdef _OPENMP
    if (n_threads < 1) n_threads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads) reduction(+ : terms)
#endif
    for (int32_t k = 0; k < n_templates; ++k) {
        double *map = (double *)malloc(sizeof(double) * n_cells);
        uint8_t *fl = (uint8_t *)malloc(n_cells);
        int32_t *cnt = (int32_t *)malloc(sizeof(int32_t) * n_cells);
        if (!map || !fl || !cnt) {
            rc = -2;
        } else {
            oracle_tfstat_map(atoms + (int64_t)k * template_stride, ld, t, n_atoms, window,
                              t0_min, dt0, N_t0, tau_min, dtau, N_tau, min_atoms, map, fl,
                              NULL, cnt, 1);
            oracle_tfstat_marginalise(map, fl, N_t0, N_tau, &out[k]);
            for (int64_t i = 0; i < n_cells; ++i) terms += cnt[i];
        }
        free(map);
        free(fl);
        free(cnt);
    }
    if (out_terms) *out_terms = terms;
    return rc;
}

/* ---------------------------------------------------------------------------------------
 * General windows on explicit grids.
 *
 * "Different window functions for the amplitude evolution could also be considered, and would
 * generically follow the GPU kernel grid setup and timing model for the exponential window"
 * (PAPER.md:192), and the {t0, tau} grid may have "a coarser or even variable sampling"
 * (PAPER.md:74).  The definition is the same cell by cell, with
 *   - t0_grid[m], tau_grid[n]: explicit integer-second arrays, any order, tau >= 1;
 *   - support = sup_num / sup_den (in units of tau): atom alpha is in the window iff
 *       t0 <= t_alpha  and  (t_alpha - t0) * sup_den < sup_num * tau     (integers, half-open);
 *   - weight w(u), u = (t_alpha - t0) / tau in [0, support):
 *       kind 0 (rect) w = 1;  kind 1 (exp) w = exp(-u);
 *       kind 2 (table) w = linear interpolation of n_table >= 2 samples table[i] = w(u_i),
 *                      u_i = i * support / (n_table - 1).
 *   With (rect, 1/1) and (exp, 3/1) this is exactly eqs. (3), (4).
 * PARITY UNPINNED BY THE PAPER for the table convention (the paper names no other window): it
 * is DESIGN.md reading R17, pinned against numpy.interp and against the rect / exp special
 * cases in tests/test_oracle_pins.py.
 * --------------------------------------------------------------------------------------- */
#define ORACLE_TABLE 2

static double general_weight(int kind, double u, double support, const float *table,
                             int32_t n_table)
{
    if (kind == ORACLE_RECT) return 1.0;
    if (kind == ORACLE_EXP) return exp(-u);
    const double x = u / support * (double)(n_table - 1);
    int64_t i = (int64_t)floor(x);
    if (i < 0) i = 0;
    if (i > n_table - 2) i = n_table - 2;
    const double f = x - (double)i;
    return (double)table[i] + f * ((double)table[i + 1] - (double)table[i]);
}

int oracle_tfstat_map_general(const float *atoms, int64_t ld, const int32_t *t, int32_t n_atoms,
                              int kind, int32_t sup_num, int32_t sup_den, const float *table,
                              int32_t n_table, const int32_t *t0_grid, int32_t N_t0,
                              const int32_t *tau_grid, int32_t N_tau, int32_t min_atoms,
                              double *out_2F, uint8_t *out_flags, double *out_cond,
                              int32_t *out_cnt, int n_threads)
{
    if (!atoms || !t || n_atoms < 1 || ld < n_atoms || !t0_grid || !tau_grid || N_t0 < 1 ||
        N_tau < 1 || !out_2F || sup_num < 1 || sup_den < 1)
        return -1;
    if (kind != ORACLE_RECT && kind != ORACLE_EXP && kind != ORACLE_TABLE) return -1;
    if (kind == ORACLE_TABLE && (!table || n_table < 2)) return -1;
    for (int32_t n = 0; n < N_tau; ++n)
        if (tau_grid[n] < 1) return -1;
    const float *a2 = atoms, *b2 = atoms + ld, *ab = atoms + 2 * ld;
    const float *fare = atoms + 3 * ld, *faim = atoms + 4 * ld;
    const float *fbre = atoms + 5 * ld, *fbim = atoms + 6 * ld;
    const double support = (double)sup_num / (double)sup_den;
#ifdef _OPENMP
    if (n_threads < 1) n_threads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
#endif
    for (int32_t m = 0; m < N_t0; ++m) {
        for (int32_t n = 0; n < N_tau; ++n) {
            const int64_t t0 = t0_grid[m], tau = tau_grid[n];
            double A = 0, B = 0, C = 0, FaRe = 0, FaIm = 0, FbRe = 0, FbIm = 0;
            int32_t cnt = 0;
            for (int32_t al = 0; al < n_atoms; ++al) {
                const int64_t dt = (int64_t)t[al] - t0;
                if (dt < 0) continue;
                if (!(dt * sup_den < (int64_t)sup_num * tau)) continue;
                const double w =
                    general_weight(kind, (double)dt / (double)tau, support, table, n_table);
                const double w2 = w * w;
                A += w2 * (double)a2[al];
                B += w2 * (double)b2[al];
                C += w2 * (double)ab[al];
                FaRe += w * (double)fare[al];
                FaIm += w * (double)faim[al];
                FbRe += w * (double)fbre[al];
                FbIm += w * (double)fbim[al];
                cnt += 1;
            }
            const double D = A * B - C * C;
            uint8_t fl = 0;
            if (cnt < min_atoms) fl |= 1;
            if (!(D > 0.0)) fl |= 2;
            const int64_t i = (int64_t)m * N_tau + n;
            out_2F[i] = fl ? 0.0
                           : 2.0 * (B * (FaRe * FaRe + FaIm * FaIm) + A * (FbRe * FbRe + FbIm * FbIm) -
                                    2.0 * C * (FaRe * FbRe + FaIm * FbIm)) / D;
            if (out_flags) out_flags[i] = fl;
            if (out_cond) out_cond[i] = (A * B != 0.0) ? D / (A * B) : 0.0;
            if (out_cnt) out_cnt[i] = cnt;
        }
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------
 * Per-detector input.  The paper's atoms carry an index "over SFTs"
 * and the map function sums whatever atoms fall into a window; with several
 * detectors the SFTs of one time stamp contribute together.  The map entry points take atoms
 * already merged per time stamp (BASELINE.json configs: "2 detectors merged per timestamp");
 * this is that merge, written out: for every output time stamp t_out[i] and every channel,
 *     out[ch][i] = sum over detectors X, in the order given, of atoms_X[ch][j]  with t_X[j] == t_out[i]
 * in fp32 (the atoms are real32; a fixed order makes the sum reproducible to the
 * bit).  Atoms of a detector whose time stamp is not in t_out are dropped; a t_out[i] that no
 * detector has gives zeros.  PARITY UNPINNED BY THE PAPER (it does not describe the merge);
 * pinned against numpy and against the merged atom model of synth/.
 * --------------------------------------------------------------------------------------- */
int oracle_merge_detectors(const float *const *atoms_dets, const int64_t *lds,
                           const int32_t *const *t_dets, const int32_t *n_dets, int32_t n_det,
                           const int32_t *t_out, int32_t n_out, float *out_atoms, int64_t ld_out)
{
    if (!atoms_dets || !lds || !t_dets || !n_dets || n_det < 1 || !t_out || n_out < 1 ||
        !out_atoms || ld_out < n_out)
        return -1;
    for (int32_t i = 0; i < n_out; ++i) {
        for (int ch = 0; ch < 7; ++ch) {
            float acc = 0.0f;
            for (int32_t x = 0; x < n_det; ++x) {
                /* linear search: plain and obviously right; the sets are small in the tests */
                for (int32_t j = 0; j < n_dets[x]; ++j) {
                    if (t_dets[x][j] == t_out[i]) {
                        acc += atoms_dets[x][ch * lds[x] + j];
                        break;
                    }
                }
            }
            out_atoms[ch * ld_out + i] = acc;
        }
    }
    return 0;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
