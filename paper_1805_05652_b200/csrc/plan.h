// plan.h -- host-side problem plan: validation, edge-lattice, tile shapes, workspace layout.
// One function of the problem shape, used by tfstat_workspace_bytes() and by every launcher,
// so the caller-provided workspace and the kernels always agree.
#pragma once
#include <stddef.h>
#include <stdint.h>

#include "tfstat_dev.cuh"

namespace tfstat {

constexpr int64_t kMaxEdgeEntries = int64_t(1) << 22;  // 16 MiB of int32; beyond: binary search
constexpr size_t kAlign = 256;

inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

inline int64_t gcd64(int64_t a, int64_t b)
{
    while (b) {
        const int64_t r = a % b;
        a = b;
        b = r;
    }
    return a;
}

// exp direct kernel tile shapes: C cells along t0 per thread, NT tau values per CTA
struct ExpTile {
    int C;
    int NT;
    int split;  // 1: the warps of a CTA share 32 tau values and split the windows' atoms
};

// rect running-sum kernel (rect.cu): a thread owns Q rows m, m+r, ..; a CTA owns NTu residues
// x 128 / NTu row groups x seg_cols columns
struct RectRun {
    int32_t enabled;  // 0: per-cell kernel (no edge lattice / very few rows)
    int32_t tile;     // 1: direct form by tiles (rect_tile_kernel); r = row offset, NTu = column offset
    int32_t Q, r, NTu, seg_cols, n_rowtiles, n_coltiles;
    int32_t ks_lg;   // >= 0: the staged run is stored in two halves of runs of 2^ks_lg entries
    int32_t ks_cap;  // lattice points of K one CTA stages in shared memory (0: K read through L1)
};

struct Plan {
    int status;  // TFSTAT_OK or error
    int window;
    int exp_method;
    int32_t n_atoms, n_templates, min_atoms;
    int32_t rect_small;  // rectangular window: the one-launch kernel of rect.cu runs this call
    Grid grid;
    // a1 edge lattice
    int64_t g;  // lattice step (s)
    int32_t e_m, e_n;
    int64_t J;  // entries; 0 if the per-cell binary-search fallback is used
    // exp direct tiling
    ExpTile tile;
    int32_t n_mtiles, n_nblocks;
    int64_t tiles_per_template;
    // exp sliding form (exp_scan.cu): t0 segments per (template, tau block)
    int32_t n_segs, seg_len;
    int32_t slide_tpc;  // templates per CTA (1, 2, 4): they share the weights
    int32_t slide_rt;   // (always 1: kept for the launchers)
    int32_t win_rt, win_tpc;  // exp_window_kernel: tau values per thread, templates per CTA
    int32_t win_nt;           // ... and threads per CTA (64 or 128; one tau per thread: 64)
    // exp_moment_kernel: tau indices [mom_n16, mom_n32) in groups of 16, [mom_n32, mom_n64) in
    // groups of 32, [mom_n64, N_tau) in groups of 64; [0, mom_n16) stay with exp_window_kernel
    // (all = N_tau: no grouped sums at all)
    int32_t mom_n16, mom_n32, mom_n64;
    // rect / marginalise tiling
    int32_t cell_blocks_per_template;
    RectRun rect;
    // workspace layout (byte offsets)
    size_t off_lo, off_edge, off_partials, off_prefix, off_tot, off_flags, off_steps, off_pack,
        off_w0, bytes;
    int32_t n_pad;  // exp: atoms per template in the packed records (pack.cu), padded
    size_t flags_bytes;  // rect: scan flags the bounds kernel (or a memset) zeroes
    int64_t partials_per_template;
    cudaEvent_t ev_main_begin, ev_main_end;  // optional profiling hooks (tfstat_opts)
    unsigned long long *stats;               // optional device work counters (tfstat_opts)
};

Plan make_plan(int window, int32_t n_atoms, int32_t n_templates, int32_t t0_min, int32_t dt0,
               int32_t N_t0, int32_t tau_min, int32_t dtau, int32_t N_tau,
               const tfstat_opts *opts);

// launchers -------------------------------------------------------------------------------
cudaError_t launch_bounds(const Plan &pl, const int32_t *t_atoms, void *ws, cudaStream_t st);
cudaError_t launch_validate_timestamps(const int32_t *t_atoms, int32_t n_atoms,
                                       int32_t *out_first_bad, cudaStream_t st);
int rect_run_threads(const Plan &pl);
cudaError_t launch_count_terms(const Plan &pl, const Bounds &b, int64_t *out_terms,
                               cudaStream_t st);
cudaError_t launch_pack(const Plan &pl, const Problem &pr, void *packed, cudaStream_t st);
cudaError_t launch_exp_direct(const Plan &pl, const Problem &pr, const void *packed,
                              Partial *partials, cudaStream_t st);
RectRun plan_rect_run(const Grid &g, int32_t e_m, int32_t e_n, int64_t J, int32_t n_templates,
                      int32_t q_override, int32_t seg_override);
int rect_scan_blocks(int32_t n_atoms);
bool rect_small_applies(int32_t n_atoms, int32_t n_templates, int64_t cells);
cudaError_t launch_rect_small(const Plan &pl, const Problem &pr, cudaStream_t st);
cudaError_t launch_rect(const Plan &pl, const Problem &pr, double *prefix, double *agg,
                        int32_t *flags, void *steps, Partial *partials, cudaStream_t st);
cudaError_t launch_exp_scan(const Plan &pl, const Problem &pr, const void *packed, void *w0,
                            Partial *partials, cudaStream_t st);
cudaError_t launch_finalize(const Partial *partials, int64_t partials_per_template,
                            int32_t n_templates, int32_t N_tau, tfstat_result *out,
                            cudaStream_t st);
cudaError_t launch_marginalise(const float *map, const uint8_t *flags, int64_t n_cells,
                               int32_t N_tau, Partial *partials, int32_t n_blocks,
                               tfstat_result *out, cudaStream_t st);
int32_t marginalise_blocks(int64_t n_cells);
cudaError_t launch_merge(const float *const *atoms, const int64_t *tstrides, const int64_t *lds,
                         const int32_t *const *ts, const int32_t *ns, int32_t n_det,
                         int32_t n_templates, const int32_t *t_out, int32_t n_out, float *out,
                         int64_t tstride_out, int64_t ld_out, cudaStream_t st);
int32_t general_partials(int32_t N_t0, int32_t N_tau);
cudaError_t launch_general(const float *atoms, int64_t ld, const int32_t *t_atoms, int32_t n_atoms,
                           const tfstat_window &w, const int32_t *t0_grid, int32_t N_t0,
                           const int32_t *tau_grid, int32_t N_tau, int32_t min_atoms,
                           float *out_map, uint8_t *out_flags, Partial *partials,
                           int32_t *n_partials, int32_t ct_override, cudaStream_t st);

inline Bounds make_bounds(const Plan &pl, const int32_t *t_atoms, void *ws)
{
    Bounds b;
    b.t = t_atoms;
    b.n_atoms = pl.n_atoms;
    b.lo = reinterpret_cast<const int32_t *>(static_cast<char *>(ws) + pl.off_lo);
    b.edge = pl.J > 0 ? reinterpret_cast<const int32_t *>(static_cast<char *>(ws) + pl.off_edge)
                      : nullptr;
    b.e_m = pl.e_m;
    b.e_n = pl.e_n;
    b.J = (int32_t)pl.J;
    return b;
}

}  // namespace tfstat
