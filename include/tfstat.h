/*
 * tfstat.h -- C ABI of libtfstat: the transient F-statistic map on NVIDIA B200 (sm_100a).
 *
 * The operation is the one stated in Keitel & Ashton 2018 (arXiv:1805.05652), section 3
 * (PAPER.md:88): "atoms + window type + {t0, tau} grid -> F_mn", eq. (8), with
 * the per-cell statistic of eq. (7) evaluated on window-weighted partial sums
 * of the atoms, windows (3)/(4), followed by the marginalisation of the map
 * (eq. (5); c_marg footnote PAPER.md:227) and batched over templates lambda
 * (PAPER.md:114, 142).  Conventions the paper leaves open are the readings R1-R16 of
 * DESIGN.md (half-open windows on atom start times, >= min_atoms atoms per cell, map stores
 * 2F, logB = log sum exp F over valid cells).
 *
 * General rules
 *  - Pointers are DEVICE pointers unless the parameter name ends in `_host` (or the function
 *    name does).  `stream` is a cudaStream_t passed as void* (NULL = default stream).
 *  - The caller owns every buffer, including `workspace`; the library allocates no device
 *    memory in the device-pointer calls, keeps no global state and is re-entrant.  Work is
 *    enqueued asynchronously on `stream`; outputs are valid once the caller synchronises.
 *  - Return value: 0 (TFSTAT_OK) or a negative tfstat_status.  Nothing throws or aborts.
 *  - Times (atom start times, t0_min, dt0, tau_min, dtau) are integer seconds relative to a
 *    caller-chosen epoch.  Window membership is decided in integers.
 *  - Atoms: 7 rows of `ld` (>= n_atoms) fp32 each, row order a2, b2, ab, Re Fa, Im Fa,
 *    Re Fb, Im Fb (the 7 x N_SFT real32 matrix of PAPER.md:88); multi-detector data merged
 *    per timestamp by the caller.  `t_atoms` strictly increasing (precondition).
 *  - Map: fp32, row-major, tau fastest: map[m*N_tau + n] = 2F(t0_min + m dt0, tau_min + n dtau)
 *    (eq. 8: m <-> t0, n <-> tau).
 *  - Degenerate cells (fewer than opts->min_atoms atoms in the window: flag bit 0; D <= 0 or
 *    NaN: flag bit 1) store 2F = 0 and are excluded from the marginals.  Empty windows and
 *    all-degenerate maps are NOT errors (the full matrix is always returned).
 */
#ifndef TFSTAT_H_
#define TFSTAT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TFSTAT_VERSION 200 /* 0.2.0: tfstat_opts starts with its own size; every call takes opts */

/* window functions, eqs. (3), (4) */
#define TFSTAT_WINDOW_RECT 0 /* w = 1 on [t0, t0 + tau)                          */
#define TFSTAT_WINDOW_EXP 1  /* w = exp(-(t - t0)/tau) on [t0, t0 + 3 tau)       */

#define TFSTAT_WINDOW_TABLE 2 /* tfstat_map_general only: w(u) tabulated, u = (t - t0)/tau    */

/* how the exponential-window sums are evaluated (tfstat_opts.exp_method) */
#define TFSTAT_EXP_AUTO 0   /* = SCAN (exact, and never slower than DIRECT: DESIGN.md 6.2) */
#define TFSTAT_EXP_DIRECT 1 /* truncated weighted sum per cell, the paper's
                               brute-force definition, register-tiled                     */
#define TFSTAT_EXP_SCAN 2   /* exact factorised, sliding form: per tau, weights
                               E_a = exp(-(t_a - t_ref)/tau) shared by all t0 (the per-cell
                               factor cancels in eq. 7); one initial window sum, then each
                               t0 step adds the entering and subtracts the leaving atoms,
                               backwards in t0; the initial sums of large tau are shared
                               between 16-64 neighbouring tau through an 8-term Taylor
                               expansion of the weight in 1/tau, truncation < 5e-9 relative
                               (csrc/exp_scan.cu)                            */

typedef enum tfstat_status {
    TFSTAT_OK = 0,
    TFSTAT_EINVAL = -1,     /* null required pointer, n_atoms < 1, N_t0 < 1, N_tau < 1, opts with
                               struct_size < 8 or reserved fields set,
                               tau_min < 1, dt0 < 1 with N_t0 > 1, dtau < 1 with N_tau > 1,
                               ld < n_atoms, unknown window/method, N_t0*N_tau >= 2^31      */
    TFSTAT_EWORKSPACE = -2, /* workspace NULL or smaller than tfstat_workspace_bytes()     */
    TFSTAT_ECUDA = -3,      /* a CUDA call failed; see tfstat_last_cuda_error()            */
    TFSTAT_EOVERFLOW = -4   /* t0_max + 3 tau_max (or any grid time) exceeds int32         */
} tfstat_status;

/* Marginals of one map (20 bytes, written on the device). */
typedef struct tfstat_result {
    float max2F;     /* max over valid cells of 2F; 0 if n_valid == 0                     */
    int32_t m;       /* t0 index of the maximum (lowest flat index m*N_tau+n on exact     */
    int32_t n;       /* ties), tau index; (-1,-1) if n_valid == 0                          */
    float logB;      /* log sum_valid exp(F), F = 2F/2; -inf if n_valid == 0               */
    int32_t n_valid; /* number of non-degenerate cells                                     */
} tfstat_result;

/* Options; a HOST pointer, the last argument of every call, NULL = defaults.
 *
 * The first field is the size of the struct THE CALLER was compiled against, so the struct can
 * grow at its end without breaking old callers: the library reads min(struct_size,
 * sizeof(tfstat_opts)) bytes and takes defaults (zeros) for the rest.  Initialise with
 * TFSTAT_OPTS_INIT (or memset to 0 and set struct_size = sizeof(tfstat_opts)); a non-NULL opts
 * with struct_size < 8 is TFSTAT_EINVAL.  The only CONVENTION of the method in here is min_atoms
 * (SURVEY.md 8(b)); everything after it selects or tunes kernels and never changes what is
 * computed beyond the rounding order. */
typedef struct tfstat_opts {
    uint32_t struct_size; /* = sizeof(tfstat_opts)                                          */
    int32_t min_atoms;  /* cells with fewer atoms are degenerate; 0 or unset -> 2
                           ("at least 2 SFTs per F_mn")                      */
    int32_t exp_method; /* TFSTAT_EXP_*                                                    */
    int32_t rect_method; /* rectangular window: 0 = auto; 1 = never the one-launch small-map
                           kernel (lattice / per-cell kernels only); 2 = the small-map kernel
                           whenever the atoms fit its shared memory (n_atoms <= 2048)          */
    int32_t tile_c;     /* tuning, 0 = chosen from the problem shape.  Direct exp kernel: t0 cells
                           per thread (1,2,4,8,16); sliding exp kernel: templates per CTA
                           (1,2,4) + 10 x (10 RT + TPC of the per-tau window-sum kernel, e.g. 422) + 1000 to
                           keep EVERY window sum with that kernel (no grouped moments); tfstat_map_general: tau cells per thread (1,2,4); lattice
                           rect kernels: rows per thread of the running-sum kernel (1, 2), or 8 =
                           the tile kernel on any grid whose lattice qualifies (auto only takes
                           it when the map has enough tiles to fill the GPU)                  */
    int32_t tile_nt;    /* tuning: threads (= tau values) per CTA (32,64,128,256); 0 = auto */
    int32_t seg_len;    /* tuning, 0 = auto.  Sliding exp kernel: t0 steps per segment; lattice
                           rect kernels: columns per CTA of the running-sum kernel (rounded up
                           to 16), < 0 = the running-sum kernel even where the tile kernel
                           (direct form) would be chosen; direct exp kernel:
                           1 = the warps of a CTA split the windows' atoms, 2 = they never do */
    int32_t reserved0;  /* must be 0 */
    /* Optional profiling hooks: cudaEvent_t handles (as void*), recorded on `stream`
     * immediately before and after the dominant kernel of the call (the window-sum +
     * closure kernel; for the rectangular window: prefix + cells kernels).  NULL = off. */
    void *ev_main_begin;
    void *ev_main_end;
    /* Optional work counters: DEVICE pointer to TFSTAT_N_STATS uint64, or NULL.  The kernels ADD
     * what they executed (the caller zeroes them): see TFSTAT_STAT_*.  Counting costs a few
     * per cent; it is meant for bench.py's roofline, not for production calls. */
    uint64_t *stats;
} tfstat_opts;
#define TFSTAT_OPTS_INIT {(uint32_t)sizeof(tfstat_opts), 0, 0, 0, 0, 0, 0, 0, NULL, NULL, NULL}

/* tfstat_opts.stats[i]: weighted (atom, cell-or-window, template) terms executed by the
 * exponential-window kernels, i.e. one weight applied to the 7 channels of one atom */
#define TFSTAT_STAT_TERMS_WINDOW 0 /* initial / direct window sums                           */
#define TFSTAT_STAT_TERMS_ENTER 1  /* sliding form: atoms entering at the low end            */
#define TFSTAT_STAT_TERMS_LEAVE 2  /* sliding form: atoms leaving at the high end            */
#define TFSTAT_STAT_TERMS_RESUM 3  /* sliding form: windows summed afresh (guard, no overlap) */
#define TFSTAT_STAT_CELLS 4        /* cells closed (eq. 7 evaluated)                          */
#define TFSTAT_STAT_REDO64 5       /* cells re-summed in fp64 (short ill-conditioned windows) */
#define TFSTAT_STAT_MOMENT 6       /* sliding form: (atom, moment, template) terms of the grouped
                                      window sums, 7 multiply-adds each                        */
#define TFSTAT_N_STATS 8

/* What the library will run for a problem shape (host-only; tfstat_plan_info()).  bench.py reads
 * its roofline's executed instruction mix from here instead of re-deriving the plan. */
#define TFSTAT_KERNEL_EXP_DIRECT 1
#define TFSTAT_KERNEL_EXP_SLIDE 2
#define TFSTAT_KERNEL_RECT_SMALL 3
#define TFSTAT_KERNEL_RECT_RUN 4   /* lattice running-sum kernel                              */
#define TFSTAT_KERNEL_RECT_CELLS 5 /* per-cell prefix differences (no lattice / few rows)     */
#define TFSTAT_KERNEL_RECT_TILE 6  /* lattice direct form, tile by tile (small lattice steps)     */
typedef struct tfstat_plan {
    uint32_t struct_size; /* in: sizeof(tfstat_plan) of the caller                           */
    int32_t kernel;       /* TFSTAT_KERNEL_* of the dominant kernel                          */
    int32_t tile_c;       /* cells (exp direct) / templates (slide) / rows (rect) per thread */
    int32_t tile_nt;      /* threads per CTA of the dominant kernel                          */
    int32_t seg_len;      /* slide: t0 steps per segment; rect run: columns per CTA          */
    int32_t n_segs;       /* slide: segments per (template, tau block); rect: column tiles   */
    int32_t n_launches;   /* kernels one tfstat_search call enqueues (results requested)     */
    int32_t lattice_J;    /* entries of the window-end lattice (0: per-cell binary search)   */
    int64_t n_ctas;       /* CTAs of the dominant kernel                                     */
    uint64_t workspace_bytes;
} tfstat_plan;

/* ---- host-only helpers (no CUDA calls) ------------------------------------------------ */
int tfstat_version(void);
const char *tfstat_strerror(int status);
/* Bytes of device workspace tfstat_map/tfstat_search need for this problem shape.
 * Returns 0 on invalid arguments. */
size_t tfstat_workspace_bytes(int window, int32_t n_atoms, int32_t n_templates, int32_t t0_min,
                              int32_t dt0, int32_t N_t0, int32_t tau_min, int32_t dtau,
                              int32_t N_tau, const tfstat_opts *opts_host);
/* Fills *info (struct_size set by the caller) for this problem shape.  0 or TFSTAT_EINVAL /
 * TFSTAT_EOVERFLOW exactly as tfstat_search would return them. */
int tfstat_plan_info(int window, int32_t n_atoms, int32_t n_templates, int32_t t0_min,
                     int32_t dt0, int32_t N_t0, int32_t tau_min, int32_t dtau, int32_t N_tau,
                     const tfstat_opts *opts_host, tfstat_plan *info);
/* cudaError_t of the last failing CUDA call made by this thread inside the library. */
int tfstat_last_cuda_error(void);

/* ---- the hot path --------------------------------------------------------------------- */

/* One template: atoms + window + grid -> full map (eq. 8).
 *   atoms      [7][ld] fp32              t_atoms   [n_atoms] int32
 *   out_map    [N_t0][N_tau] fp32 2F     out_flags [N_t0][N_tau] uint8, nullable
 *   workspace  >= tfstat_workspace_bytes(window, n_atoms, 1, grid...) bytes, 256-B aligned */
int tfstat_map(const float *atoms, int64_t ld, const int32_t *t_atoms, int32_t n_atoms,
               int window, int32_t t0_min, int32_t dt0, int32_t N_t0, int32_t tau_min,
               int32_t dtau, int32_t N_tau, float *out_map, uint8_t *out_flags,
               void *workspace, size_t workspace_bytes, void *stream,
               const tfstat_opts *opts_host);

/* Marginalise a map already in device memory: max 2F + argmax, logB, n_valid.
 *   flags nullable (NULL: every cell valid).  out: one tfstat_result on the device.
 *   workspace: >= tfstat_marginalise_workspace_bytes(N_t0, N_tau) bytes, 16-byte aligned
 *   (TFSTAT_EWORKSPACE otherwise).  opts_host: nothing in it applies yet (reserved).       */
size_t tfstat_marginalise_workspace_bytes(int32_t N_t0, int32_t N_tau);
int tfstat_marginalise(const float *map, const uint8_t *flags, int32_t N_t0, int32_t N_tau,
                       tfstat_result *out, void *workspace, size_t workspace_bytes,
                       void *stream, const tfstat_opts *opts_host);

/* tfstat_marginalise WITHOUT a workspace and without any allocation, for callers that cannot
 * call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
 * the scratch is a static __device__ array inside the library (37 888 bytes on every GPU that
 * loads it).  Same kernels, same results as tfstat_marginalise, bit for bit.
 *   Maximum: N_t0 * N_tau <= tfstat_marginalise_static_max_cells() = 2^31 - 1 (the scratch serves
 *   every such map); beyond it TFSTAT_EINVAL, and TFSTAT_EWORKSPACE should a map ever need more
 *   scratch records than the array holds.
 *   The device that is current at the call must be the one `map`, `flags`, `out` and `stream`
 *   belong to.  Every call on a device shares the one array: calls ordered on a stream are safe,
 *   calls that OVERLAP on the GPU (other streams, concurrent graph replays) race on it.  Nothing
 *   in it needs clearing between calls.  The first call on a device looks the array's address
 *   up (cudaGetSymbolAddress: no allocation); make it outside graph capture. */
size_t tfstat_marginalise_static_max_cells(void);
int tfstat_marginalise_static(const float *map, const uint8_t *flags, int32_t N_t0,
                              int32_t N_tau, tfstat_result *out, void *stream);

/* Batched search over n_templates independent atom sets that share timestamps and grid;
 * map evaluation, cell closure and marginalisation fused, so only n_templates results reach
 * memory unless out_maps is given (eq. 5).
 *   atoms      template k, row r, atom i at atoms[k*template_stride + r*ld + i]
 *   out        [n_templates] tfstat_result
 *   out_maps   nullable; [n_templates][N_t0][N_tau] fp32, streamed as computed
 *   out_flags  nullable; same shape, uint8                                                */
int tfstat_search(const float *atoms, int64_t template_stride, int64_t ld,
                  const int32_t *t_atoms, int32_t n_atoms, int32_t n_templates, int window,
                  int32_t t0_min, int32_t dt0, int32_t N_t0, int32_t tau_min, int32_t dtau,
                  int32_t N_tau, tfstat_result *out, float *out_maps, uint8_t *out_flags,
                  void *workspace, size_t workspace_bytes, void *stream,
                  const tfstat_opts *opts_host);

/* Number of (cell, atom-in-window) terms of the grid, the N_sums of eqs. (A.5)/(A.6)
 * generalised to gaps: sum over cells of the atoms in
 * [t0, t0 + k tau), k = 1 (rect) or 3 (exp).  *out_terms is a DEVICE int64.
 *   workspace: >= tfstat_workspace_bytes(window, n_atoms, 1, grid...) bytes.               */
int tfstat_count_terms(const int32_t *t_atoms, int32_t n_atoms, int window, int32_t t0_min,
                       int32_t dt0, int32_t N_t0, int32_t tau_min, int32_t dtau,
                       int32_t N_tau, int64_t *out_terms, void *workspace,
                       size_t workspace_bytes, void *stream, const tfstat_opts *opts_host);

/* Opt-in check of the precondition "t_atoms strictly increasing" (gaps are fine, PAPER.md:90;
 * unsorted or duplicate time stamps are not: every kernel finds its windows by binary search).
 * The data lives on the device, so the answer does too:
 *   *out_first_bad (DEVICE int32) = smallest i >= 1 with t_atoms[i] <= t_atoms[i-1], or -1.
 * Errors: TFSTAT_EINVAL (null pointer, n_atoms < 1). */
int tfstat_validate_timestamps(const int32_t *t_atoms, int32_t n_atoms, int32_t *out_first_bad,
                               void *stream, const tfstat_opts *opts_host);

/* ---- general windows on explicit grids ------------------------------------------------ */

/* A window function for tfstat_map_general (a HOST struct; `table` is a DEVICE pointer).
 * "Different window functions for the amplitude evolution could also be considered, and would
 * generically follow the GPU kernel grid setup ... for the exponential window".
 *   support = support_num / support_den, in units of tau: atom a is in the window iff
 *     t0 <= t_a  and  (t_a - t0) * support_den < support_num * tau   (integers, half-open);
 *   weight w(u), u = (t_a - t0)/tau in [0, support), applied as w on Fa, Fb and w^2 on
 *   a2, b2, ab:   TFSTAT_WINDOW_RECT  w = 1          (support 1/1: eq. 3)
 *                 TFSTAT_WINDOW_EXP   w = exp(-u)    (support 3/1: eq. 4)
 *                 TFSTAT_WINDOW_TABLE w = linear interpolation of n_table >= 2 fp32 samples
 *                                     table[i] = w(i * support / (n_table - 1)).            */
typedef struct tfstat_window {
    int32_t kind;
    int32_t support_num, support_den; /* both >= 1 */
    int32_t n_table;                  /* TABLE only */
    const float *table;               /* TABLE only; device memory, n_table floats */
} tfstat_window;

/* Map (and / or marginals) for a general window on EXPLICIT grids: t0_grid[N_t0] and
 * tau_grid[N_tau] are DEVICE int32 arrays of seconds in any order ("a coarser or even variable
 * sampling is also possible"); map[m*N_tau + n] = 2F(t0_grid[m], tau_grid[n]).
 * Every cell is the direct truncated sum.  Entries tau_grid[n] < 1 give
 * degenerate cells (flags 3), not an error (the arrays live on the device).
 *   out_map, out_flags, out: each nullable, at least one of out_map / out required.
 *   workspace: >= tfstat_general_workspace_bytes(N_t0, N_tau) bytes, 256-B aligned.
 *   opts_host: min_atoms, and tile_c (tuning: tau cells per thread, 1 / 2 / 4; 0 = auto).     */
size_t tfstat_general_workspace_bytes(int32_t N_t0, int32_t N_tau);
int tfstat_map_general(const float *atoms, int64_t ld, const int32_t *t_atoms, int32_t n_atoms,
                       const tfstat_window *window_host, const int32_t *t0_grid, int32_t N_t0,
                       const int32_t *tau_grid, int32_t N_tau, float *out_map,
                       uint8_t *out_flags, tfstat_result *out, void *workspace,
                       size_t workspace_bytes, void *stream, const tfstat_opts *opts_host);

/* ---- per-detector input ----------------------------------------------------------------- */

#define TFSTAT_MAX_DETECTORS 8

/* Merge per-detector atoms onto one set of time stamps (atoms are indexed "over SFTs",
 * PAPER.md:65; the map entry points above take them merged per time stamp):
 *   out[k][ch][i] = sum over detectors X = 0..n_det-1, in this order, of atoms_X[k][ch][j]
 *                   with t_X[j] == t_out[i]                (fp32; reproducible to the bit)
 * Atoms of a detector whose time stamp is not in t_out are dropped; a t_out[i] that no detector
 * has gives zeros.  The caller chooses t_out (normally the sorted union of the t_X).
 *   atoms_dets, t_dets: HOST arrays of n_det DEVICE pointers; atoms_dets[X] is laid out like the
 *   atoms of tfstat_search with template_strides[X], lds[X] (HOST arrays); t_dets[X] has
 *   n_atoms_dets[X] strictly increasing int32 time stamps, shared by all templates.
 *   t_out: DEVICE [n_out] strictly increasing; out_atoms: DEVICE [n_templates][7][ld_out].
 * Errors: TFSTAT_EINVAL (null pointers, n_det outside 1..TFSTAT_MAX_DETECTORS, sizes < 1,
 * ld < n).                                                                                  */
int tfstat_merge_detectors(const float *const *atoms_dets, const int64_t *template_strides,
                           const int64_t *lds, const int32_t *const *t_dets,
                           const int32_t *n_atoms_dets, int32_t n_det, int32_t n_templates,
                           const int32_t *t_out, int32_t n_out, float *out_atoms,
                           int64_t template_stride_out, int64_t ld_out, void *stream,
                           const tfstat_opts *opts_host);

/* ---- end-to-end entry point with HOST buffers ----------------------------------------- */

/* tfstat_search on host memory: copies atoms host->device in template chunks on internal
 * streams (overlapped with compute), runs the fused search, copies results (and maps, if
 * asked) device->host, and returns after everything has completed.  Host buffers should be
 * page-locked for the copies to overlap.  This is the paper's per-template copy-in / kernel /
 * copy-out without the per-template round trip.
 *   atoms_host, t_atoms_host, out_host, out_maps_host (nullable): HOST pointers, layouts as
 *   in tfstat_search.
 *   device_scratch: DEVICE buffer of device_scratch_bytes bytes (256-B aligned; not in use by
 *   work still running on any stream of the caller: the library uses streams of its own) that holds the
 *   double-buffered chunks, the workspace and the results.  Any size from one template's worth
 *   up works (smaller => more, smaller chunks); tfstat_search_host_scratch_bytes() gives the
 *   size for the preferred chunks.  NULL: the library cudaMallocs up to
 *   device_scratch_bytes (0 = 2 GiB) itself and frees it before returning -- convenient, but
 *   cudaFree can stall for ~100 ms, so callers in a loop should pass their own buffer.
 *   Errors: TFSTAT_EWORKSPACE if a given scratch is misaligned or too small for one template. */
int tfstat_search_host(const float *atoms_host, int64_t template_stride, int64_t ld,
                       const int32_t *t_atoms_host, int32_t n_atoms, int32_t n_templates,
                       int window, int32_t t0_min, int32_t dt0, int32_t N_t0, int32_t tau_min,
                       int32_t dtau, int32_t N_tau, tfstat_result *out_host,
                       float *out_maps_host, void *device_scratch, size_t device_scratch_bytes,
                       const tfstat_opts *opts_host);
/* Host-only: scratch size for the preferred chunks (n_templates / 4, clamped to 256..1024
 * templates); 0 on invalid input. */
size_t tfstat_search_host_scratch_bytes(int64_t template_stride, int32_t n_atoms,
                                        int32_t n_templates, int window, int32_t t0_min,
                                        int32_t dt0, int32_t N_t0, int32_t tau_min, int32_t dtau,
                                        int32_t N_tau, int want_maps,
                                        const tfstat_opts *opts_host);

#ifdef __cplusplus
}
#endif
#endif /* TFSTAT_H_ */
