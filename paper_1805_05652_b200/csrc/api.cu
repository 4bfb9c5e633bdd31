// api.cu -- the C ABI of include/tfstat.h: argument validation, the problem plan (workspace
// layout, tile shapes) and the launch sequences.  No arithmetic of the method lives here.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "plan.h"

namespace tfstat {

static thread_local int g_last_cuda_error = 0;

static int cuda_fail(cudaError_t e)
{
    g_last_cuda_error = (int)e;
    return TFSTAT_ECUDA;
}
#define TF_CUDA(call)                                   \
    do {                                                \
        cudaError_t e__ = (call);                       \
        if (e__ != cudaSuccess) return cuda_fail(e__);  \
    } while (0)

// tfstat_opts as the caller sees it -> the library's own, complete copy: min(struct_size,
// sizeof) bytes are the caller's, the rest defaults (include/tfstat.h)
struct OptsIn {
    tfstat_opts o;
    bool ok;
    explicit OptsIn(const tfstat_opts *in)
    {
        std::memset(&o, 0, sizeof(o));
        o.struct_size = (uint32_t)sizeof(o);
        ok = true;
        if (!in) return;
        if (in->struct_size < 8) {
            ok = false;
            return;
        }
        std::memcpy(&o, in, std::min<size_t>(in->struct_size, sizeof(o)));
        o.struct_size = (uint32_t)sizeof(o);
        if (o.reserved0 != 0) ok = false;
    }
};

Plan make_plan(int window, int32_t n_atoms, int32_t n_templates, int32_t t0_min, int32_t dt0,
               int32_t N_t0, int32_t tau_min, int32_t dtau, int32_t N_tau,
               const tfstat_opts *opts)
{
    Plan pl;
    std::memset(&pl, 0, sizeof(pl));
    pl.status = TFSTAT_EINVAL;
    if (window != TFSTAT_WINDOW_RECT && window != TFSTAT_WINDOW_EXP) return pl;
    if (n_atoms < 1 || n_templates < 1 || N_t0 < 1 || N_tau < 1 || tau_min < 1) return pl;
    if ((N_t0 > 1 && dt0 < 1) || (N_tau > 1 && dtau < 1)) return pl;
    if ((int64_t)N_t0 * N_tau >= (int64_t(1) << 31)) return pl;
    int method = opts ? opts->exp_method : TFSTAT_EXP_AUTO;
    // AUTO = the exact sliding form: same accuracy as the direct sum against the oracle (worst
    // |d 2F| 0.02 x tolerance for both on configs 2-5 and on 30-80 % gap cases) and never slower
    // in any shape measured (1.0x at N_t0 = 16 ... 33x on config 5); DESIGN.md 6.2
    if (method == TFSTAT_EXP_AUTO) method = TFSTAT_EXP_SCAN;
    if (method != TFSTAT_EXP_DIRECT && method != TFSTAT_EXP_SCAN) return pl;
    const int64_t k = window == TFSTAT_WINDOW_EXP ? 3 : 1;
    const int64_t t0_max = (int64_t)t0_min + (int64_t)(N_t0 - 1) * (N_t0 > 1 ? dt0 : 0);
    const int64_t tau_max = (int64_t)tau_min + (int64_t)(N_tau - 1) * (N_tau > 1 ? dtau : 0);
    if (t0_max + k * tau_max > INT32_MAX || t0_max > INT32_MAX || tau_max > INT32_MAX) {
        pl.status = TFSTAT_EOVERFLOW;
        return pl;
    }
    pl.window = window;
    pl.exp_method = method;
    pl.n_atoms = n_atoms;
    pl.n_templates = n_templates;
    pl.min_atoms = (opts && opts->min_atoms > 0) ? opts->min_atoms : 2;
    pl.ev_main_begin = opts ? static_cast<cudaEvent_t>(opts->ev_main_begin) : nullptr;
    pl.ev_main_end = opts ? static_cast<cudaEvent_t>(opts->ev_main_end) : nullptr;
    pl.stats = opts ? reinterpret_cast<unsigned long long *>(opts->stats) : nullptr;
    pl.grid.t0_min = t0_min;
    pl.grid.dt0 = N_t0 > 1 ? dt0 : 0;
    pl.grid.N_t0 = N_t0;
    pl.grid.tau_min = tau_min;
    pl.grid.dtau = N_tau > 1 ? dtau : 0;
    pl.grid.N_tau = N_tau;
    pl.grid.k = (int32_t)k;

    // a1 edge lattice: every window end t0_m + k tau_n sits on base + j g
    const int64_t sa = pl.grid.dt0, sb = k * pl.grid.dtau;
    int64_t g = gcd64(sa, sb);
    if (g == 0) g = 1;
    pl.g = g;
    pl.e_m = (int32_t)(sa / g);
    pl.e_n = (int32_t)(sb / g);
    pl.J = (int64_t)(N_t0 - 1) * pl.e_m + (int64_t)(N_tau - 1) * pl.e_n + 1;
    if (pl.J > kMaxEdgeEntries) {
        pl.J = 0;  // per-cell binary search instead
        pl.e_m = pl.e_n = 0;
    }

    // exp direct tile shape: largest tile that still yields a few waves of CTAs on 148 SMs
    const int64_t cells = (int64_t)N_t0 * N_tau;
    // C = 8 executes 7.25 FP32 ops per term, C = 4 7.5 (3 % more) but gives twice the CTAs: take
    // C = 8 only when it still fills 148 SMs x 4 resident CTAs about 8 times over (measured on
    // B200: configs 2 and 3, under one wave at C = 8, are 25-30 % faster at C = 4)
    auto n_ctas = [&](int c, int nt) {
        return (int64_t)((N_t0 + c - 1) / c) * ((N_tau + nt - 1) / nt) * n_templates;
    };
    const int64_t wave = 148 * 4;
    int C = n_ctas(8, 128) >= 8 * wave ? 8 : n_ctas(4, 64) >= wave ? 4 : 2;
    // one weight per t0 tile (exp_direct.cu): the per-cell factor exp(-(c dt0)/tau) that the
    // closure is invariant to must stay well inside fp32 range
    while (C > 1 && (int64_t)(C - 1) * pl.grid.dt0 > (int64_t)8 * tau_min) C >>= 1;
    pl.tile = ExpTile{C, n_ctas(C, 128) >= wave ? 128 : 64, 0};
    // Too few CTAs to fill the GPU several times over (a single map): the warps of a CTA split
    // the windows' atoms instead of the tau values (exp_direct.cu, SPLIT): 32 tau per CTA, four
    // times the CTAs, a quarter of the critical path each.  C from the same rule on that grid.
    if (n_ctas(8, 128) < 8 * wave) {
        // (measured on B200, single maps: config 2 C = 8 / 4 / 2: 166 / 169 / 190 us; config 3:
        // 528 / 563 / 647 us; unsplit C = 4: 170 / 593 us)
        int Cs = n_ctas(8, 32) >= 2 * wave ? 8 : n_ctas(4, 32) >= wave ? 4 : 2;
        while (Cs > 1 && (int64_t)(Cs - 1) * pl.grid.dt0 > (int64_t)8 * tau_min) Cs >>= 1;
        pl.tile = ExpTile{Cs, 128, 1};
    }
    if (opts && opts->tile_c && !(window == TFSTAT_WINDOW_EXP && method == TFSTAT_EXP_SCAN)) {
        const int c = opts->tile_c;
        if (c != 1 && c != 2 && c != 4 && c != 8 && c != 16) return pl;
        pl.tile.C = c;
        // the underflow guard above also binds a requested tile: the weight shared by a t0 tile
        // drops by exp(-(C-1) dt0 / tau_min) across it
        while (pl.tile.C > 1 && (int64_t)(pl.tile.C - 1) * pl.grid.dt0 > (int64_t)8 * tau_min)
            pl.tile.C >>= 1;
    }
    if (opts && opts->tile_nt) {
        const int nt = opts->tile_nt;
        if (nt != 32 && nt != 64 && nt != 128 && nt != 256) return pl;
        pl.tile.NT = nt;
    }
    if (opts && opts->seg_len && window == TFSTAT_WINDOW_EXP && method == TFSTAT_EXP_DIRECT) {
        if (opts->seg_len != 1 && opts->seg_len != 2) return pl;
        pl.tile.split = opts->seg_len == 1;
    }
    if (pl.tile.C > 8 || pl.tile.NT != 128) pl.tile.split = 0;  // the split form's one shape
    const int tpb = pl.tile.split ? 32 : pl.tile.NT;  // tau values per CTA
    pl.n_mtiles = (N_t0 + pl.tile.C - 1) / pl.tile.C;
    pl.n_nblocks = (N_tau + tpb - 1) / tpb;
    pl.tiles_per_template = (int64_t)pl.n_mtiles * pl.n_nblocks;
    pl.cell_blocks_per_template = (int32_t)((cells + 255) / 256);

    const bool direct = window == TFSTAT_WINDOW_EXP && method == TFSTAT_EXP_DIRECT;
    const bool slide = window == TFSTAT_WINDOW_EXP && method == TFSTAT_EXP_SCAN;
    if (slide) {
        // sliding form: one thread per tau, NT tau per CTA, t0 cut into segments only when
        // (templates x tau blocks) alone cannot fill 148 SMs with ~16 warps each
        int NT = 128;
        const int64_t want_warps = 148 * 16;
        while (NT > 32 && (int64_t)n_templates * ((N_tau + NT - 1) / NT) * (NT / 32) < want_warps)
            NT >>= 1;
        if (opts && opts->tile_nt) {
            if (opts->tile_nt != 32 && opts->tile_nt != 64 && opts->tile_nt != 128) return pl;
            NT = opts->tile_nt;
        }
        pl.tile.NT = NT;
        pl.n_nblocks = (N_tau + NT - 1) / NT;
        const int64_t warps = (int64_t)n_templates * pl.n_nblocks * (NT / 32);
        int64_t segs = (want_warps + warps - 1) / warps;
        const int64_t max_segs = (N_t0 + 31) / 32;  // a segment holds at least 32 t0 steps
        if (segs > max_segs) segs = max_segs;
        if (segs < 1) segs = 1;
        int32_t len = (int32_t)((N_t0 + segs - 1) / segs);
        if (opts && opts->seg_len > 0) len = opts->seg_len < N_t0 ? opts->seg_len : N_t0;
        pl.seg_len = len;
        pl.n_segs = (N_t0 + len - 1) / len;
        // slide kernel: templates per CTA (they share the weights): 2 while that still leaves the
        // GPU ~16 CTAs per SM
        const int64_t ctas1 = (int64_t)n_templates * pl.n_nblocks * pl.n_segs;
        pl.slide_tpc = (n_templates >= 2 && ctas1 / 2 >= 148 * 16) ? 2 : 1;
        // 4 where the batch is large (3 CTAs of 168 registers per SM; config 4: 7 % faster than 2)
        if (NT == 128 && n_templates >= 4 && ctas1 / 4 >= 148 * 24) pl.slide_tpc = 4;
        pl.slide_rt = 1;
        // grouped window sums (exp_moment_kernel): a group of R neighbouring tau shares 8 moments
        // while z = (window length) x (half width of the group in 1/tau) <= 1.5 (R - 1) dtau / tau
        // stays below 0.17 (exp_scan.cu: the truncation bound); R = 64 above that tau, R = 32 above half of
        // it, R = 16 above a quarter, the per-tau recurrence below.  Regions shorter than one group are not worth a launch.
        bool moments = n_templates >= 2;
        int tile_code = opts ? opts->tile_c : 0;
        if (tile_code >= 1000) moments = false, tile_code -= 1000;  // 1000 + ...: never
        pl.mom_n16 = pl.mom_n32 = pl.mom_n64 = N_tau;
        if (moments) {
            auto first_n = [&](int R) {  // first tau index with tau >= 1.5 (R - 1) dtau / 0.17
                const double tau_R = 1.5 * (R - 1) * (double)pl.grid.dtau / 0.17;
                const double x = std::ceil((tau_R - (double)pl.grid.tau_min) / (double)pl.grid.dtau);
                return (int32_t)std::min<double>(std::max(x, 0.0), (double)N_tau);
            };
            pl.mom_n64 = first_n(64);
            pl.mom_n32 = first_n(32);
            pl.mom_n16 = first_n(16);
            if (N_tau - pl.mom_n64 < 64) pl.mom_n64 = N_tau;
            if (pl.mom_n64 - pl.mom_n32 < 32) pl.mom_n32 = pl.mom_n64;
            if (pl.mom_n32 - pl.mom_n16 < 16) pl.mom_n16 = pl.mom_n32;
        }
        // per-tau window kernel (exp_window_kernel) for the tau indices [0, mom_n16): RT tau values
        // per thread x TPC templates per CTA share every broadcast load of an atom.  Of the tiles
        // that give the GPU ~8 warps per SM, the one with the least cost: slots (the range rounded
        // up to whole CTAs) x the relative cost of a slot (RT = 4 1.0, RT = 2 1.15, one tau per
        // thread 1.6); short ranges -- what the grouped sums leave over -- take 64-thread CTAs.
        {
            const int n_lim = pl.mom_n16 > 0 ? pl.mom_n16 : 1;
            const int tpc = n_templates >= 2 ? 2 : 1;
            auto warps = [&](int nt, int rt, int t) {
                return (int64_t)((n_lim + nt * rt - 1) / (nt * rt)) * pl.n_segs *
                       ((n_templates + t - 1) / t) * (nt / 32);
            };
            auto cost = [&](int nt, int rt, double per_slot) {
                const int64_t b = (int64_t)nt * rt;
                return (double)((n_lim + b - 1) / b * b) * per_slot;
            };
            pl.win_nt = 64, pl.win_rt = 1, pl.win_tpc = warps(64, 1, tpc) >= 148 * 8 ? tpc : 1;
            double best = cost(64, 1, 1.6);
            const int cand[4][2] = {{64, 2}, {128, 2}, {64, 4}, {128, 4}};
            for (const auto &cd : cand) {
                const double cst = cost(cd[0], cd[1], cd[1] == 2 ? 1.15 : 1.0);
                if (warps(cd[0], cd[1], tpc) >= 148 * 8 && cst <= best)
                    pl.win_nt = cd[0], pl.win_rt = cd[1], pl.win_tpc = tpc, best = cst;
            }
        }
        if (tile_code) {  // TPC of the slide kernel + 10 x (RT TPC code of the window kernel)
            const int c = tile_code, w = c / 10, sl = c % 10;
            if (sl != 1 && sl != 2 && sl != 4) return pl;
            if (w != 0 && w != 11 && w != 12 && w != 21 && w != 22 && w != 41 && w != 42) return pl;
            pl.slide_tpc = (sl == 4 && pl.tile.NT != 128) ? 2 : sl;  // 4: 128-thread CTAs only
            if (w) {  // (a requested tile keeps 128-thread CTAs, but one tau per thread has 64)
                pl.win_rt = w / 10, pl.win_tpc = w % 10;
                pl.win_nt = pl.win_rt == 1 ? 64 : 128;
            }
        }
    }
    if (window == TFSTAT_WINDOW_RECT) {
        const int rm = opts ? opts->rect_method : 0;
        if (rm < 0 || rm > 2) return pl;
        pl.rect_small = rm == 1   ? 0
                        : rm == 2 ? (n_atoms <= 2048)
                                  : rect_small_applies(n_atoms, n_templates, cells);
    }
    if (window == TFSTAT_WINDOW_RECT)
        pl.rect = plan_rect_run(pl.grid, pl.e_m, pl.e_n, pl.J, n_templates, opts ? opts->tile_c : 0,
                                opts ? opts->seg_len : 0);
    pl.partials_per_template = direct  ? pl.tiles_per_template
                               : slide ? (int64_t)pl.n_nblocks * pl.n_segs
                               : pl.rect.enabled
                                   ? (int64_t)pl.rect.n_rowtiles * pl.rect.n_coltiles
                                   : pl.cell_blocks_per_template;
    if (pl.partials_per_template * n_templates >= (int64_t(1) << 31)) return pl;

    size_t off = 0;
    pl.off_lo = off;
    off += align_up(sizeof(int32_t) * (size_t)N_t0);
    pl.off_edge = off;
    off += align_up(sizeof(int32_t) * (size_t)pl.J);
    pl.off_partials = off;
    off += align_up(sizeof(Partial) * (size_t)pl.partials_per_template * n_templates);
    pl.off_prefix = off;
    if (window == TFSTAT_WINDOW_RECT)
        off += align_up(sizeof(double) * 8 * ((size_t)n_atoms + 1) * n_templates);
    pl.off_tot = off;
    if (window == TFSTAT_WINDOW_RECT)
        off += align_up(sizeof(double) * 8 * (size_t)rect_scan_blocks(n_atoms) * n_templates);
    pl.off_flags = off;
    pl.flags_bytes = 0;
    if (window == TFSTAT_WINDOW_RECT) {
        pl.flags_bytes = sizeof(int32_t) * 2 * (size_t)rect_scan_blocks(n_atoms) * n_templates;
        off += align_up(pl.flags_bytes);
    }
    pl.off_steps = off;
    if (window == TFSTAT_WINDOW_RECT && pl.rect.enabled)
        off += align_up((size_t)64 * (size_t)(pl.J + 1) * n_templates);
    pl.off_pack = off;
    pl.n_pad = 0;
    if (window == TFSTAT_WINDOW_EXP) {
        pl.n_pad = (int32_t)(((int64_t)n_atoms + kPackBlock - 1) / kPackBlock * kPackBlock);
        off += align_up((size_t)32 * (size_t)pl.n_pad * n_templates);
    }
    pl.off_w0 = off;  // sliding form: window sums of each segment's last t0, 32 B per (template, segment, tau)
    if (slide) off += align_up((size_t)32 * (size_t)n_templates * pl.n_segs * N_tau);
    pl.bytes = off;
    pl.status = TFSTAT_OK;
    return pl;
}

static int run_device(const Plan &pl, const float *atoms, int64_t template_stride, int64_t ld,
                      const int32_t *t_atoms, tfstat_result *out, float *out_maps,
                      uint8_t *out_flags, void *ws, cudaStream_t st, bool do_bounds)
{
    const bool small = pl.window == TFSTAT_WINDOW_RECT && pl.rect_small;
    if (small) {
        // one launch does bounds, sums, closure, marginals and the result record
    } else if (do_bounds) {
        TF_CUDA(launch_bounds(pl, t_atoms, ws, st));
    } else if (pl.flags_bytes) {
        TF_CUDA(cudaMemsetAsync(static_cast<char *>(ws) + pl.off_flags, 0, pl.flags_bytes, st));
    }
    Problem pr;
    pr.atoms = atoms;
    pr.template_stride = template_stride;
    pr.ld = ld;
    pr.n_templates = pl.n_templates;
    pr.min_atoms = pl.min_atoms;
    pr.grid = pl.grid;
    pr.bounds = make_bounds(pl, t_atoms, ws);
    pr.out = out;
    pr.out_maps = out_maps;
    pr.out_flags = out_flags;
    Partial *partials =
        out ? reinterpret_cast<Partial *>(static_cast<char *>(ws) + pl.off_partials) : nullptr;
    void *packed = static_cast<char *>(ws) + pl.off_pack;
    if (pl.window == TFSTAT_WINDOW_EXP) TF_CUDA(launch_pack(pl, pr, packed, st));
    if (pl.ev_main_begin) TF_CUDA(cudaEventRecord(pl.ev_main_begin, st));
    if (small) {
        TF_CUDA(launch_rect_small(pl, pr, st));
        if (pl.ev_main_end) TF_CUDA(cudaEventRecord(pl.ev_main_end, st));
        return TFSTAT_OK;
    }
    if (pl.window == TFSTAT_WINDOW_RECT) {
        double *prefix = reinterpret_cast<double *>(static_cast<char *>(ws) + pl.off_prefix);
        double *agg = reinterpret_cast<double *>(static_cast<char *>(ws) + pl.off_tot);
        int32_t *flags = reinterpret_cast<int32_t *>(static_cast<char *>(ws) + pl.off_flags);
        TF_CUDA(launch_rect(pl, pr, prefix, agg, flags, static_cast<char *>(ws) + pl.off_steps,
                            partials, st));
    } else if (pl.exp_method == TFSTAT_EXP_DIRECT) {
        TF_CUDA(launch_exp_direct(pl, pr, packed, partials, st));
    } else {
        TF_CUDA(launch_exp_scan(pl, pr, packed, static_cast<char *>(ws) + pl.off_w0, partials, st));
    }
    if (pl.ev_main_end) TF_CUDA(cudaEventRecord(pl.ev_main_end, st));
    if (out)
        TF_CUDA(launch_finalize(partials, pl.partials_per_template, pl.n_templates,
                                pl.grid.N_tau, out, st));
    return TFSTAT_OK;
}

// Templates per chunk of tfstat_search_host: about four chunks per call (so that the copies
// overlap the compute), at least 256 and at most 1024 templates (a chunk must still fill the GPU
// with the sliding form, which runs up to 4 templates per CTA).
static int32_t host_chunk_templates(int32_t n_templates)
{
    return std::min<int32_t>(n_templates, std::max<int32_t>(256, std::min<int32_t>(1024, n_templates / 4)));
}

// Plans of tfstat_search_host for chunks of Tc templates: the full chunks' plan, the plan of the
// ragged last chunk (tile shapes depend on the number of templates, so it may need MORE
// workspace than a full chunk), and the workspace that serves both.
static int plan_host_chunks(int window, int32_t n_atoms, int32_t n_templates, int32_t Tc,
                            int32_t t0_min, int32_t dt0, int32_t N_t0, int32_t tau_min,
                            int32_t dtau, int32_t N_tau, const tfstat_opts *opts, Plan &pl,
                            Plan &pl_last, size_t &ws_bytes)
{
    pl = make_plan(window, n_atoms, Tc, t0_min, dt0, N_t0, tau_min, dtau, N_tau, opts);
    if (pl.status != TFSTAT_OK) return pl.status;
    pl_last = pl;
    const int32_t rem = n_templates % Tc;
    if (rem != 0) {
        pl_last = make_plan(window, n_atoms, rem, t0_min, dt0, N_t0, tau_min, dtau, N_tau, opts);
        if (pl_last.status != TFSTAT_OK) return pl_last.status;
    }
    ws_bytes = align_up(std::max(std::max(pl.bytes, pl_last.bytes), kAlign));
    return TFSTAT_OK;
}

}  // namespace tfstat

using namespace tfstat;

extern "C" {

int tfstat_version(void) { return TFSTAT_VERSION; }

const char *tfstat_strerror(int status)
{
    switch (status) {
    case TFSTAT_OK: return "ok";
    case TFSTAT_EINVAL: return "invalid argument";
    case TFSTAT_EWORKSPACE: return "workspace missing or too small";
    case TFSTAT_ECUDA: return "CUDA error (see tfstat_last_cuda_error)";
    case TFSTAT_EOVERFLOW: return "grid times exceed int32";
    default: return "unknown status";
    }
}

int tfstat_last_cuda_error(void) { return g_last_cuda_error; }

size_t tfstat_workspace_bytes(int window, int32_t n_atoms, int32_t n_templates, int32_t t0_min,
                              int32_t dt0, int32_t N_t0, int32_t tau_min, int32_t dtau,
                              int32_t N_tau, const tfstat_opts *opts_host)
{
    const OptsIn oi(opts_host);
    if (!oi.ok) return 0;
    const Plan pl = make_plan(window, n_atoms, n_templates, t0_min, dt0, N_t0, tau_min, dtau,
                              N_tau, &oi.o);
    return pl.status == TFSTAT_OK ? std::max(pl.bytes, kAlign) : 0;
}

int tfstat_plan_info(int window, int32_t n_atoms, int32_t n_templates, int32_t t0_min,
                     int32_t dt0, int32_t N_t0, int32_t tau_min, int32_t dtau, int32_t N_tau,
                     const tfstat_opts *opts_host, tfstat_plan *info)
{
    if (!info || info->struct_size < 8) return TFSTAT_EINVAL;
    const OptsIn oi(opts_host);
    if (!oi.ok) return TFSTAT_EINVAL;
    const Plan pl = make_plan(window, n_atoms, n_templates, t0_min, dt0, N_t0, tau_min, dtau,
                              N_tau, &oi.o);
    if (pl.status != TFSTAT_OK) return pl.status;
    tfstat_plan p;
    std::memset(&p, 0, sizeof(p));
    p.lattice_J = (int32_t)pl.J;
    p.workspace_bytes = std::max(pl.bytes, kAlign);
    if (window == TFSTAT_WINDOW_EXP && pl.exp_method == TFSTAT_EXP_DIRECT) {
        p.kernel = TFSTAT_KERNEL_EXP_DIRECT;
        p.tile_c = pl.tile.C;
        p.tile_nt = pl.tile.NT;
        p.n_ctas = pl.tiles_per_template * n_templates;
        p.n_launches = 4;  // bounds, pack, sums + closure + marginals, finalize
    } else if (window == TFSTAT_WINDOW_EXP) {
        p.kernel = TFSTAT_KERNEL_EXP_SLIDE;
        p.tile_c = pl.slide_tpc + 10 * (10 * pl.win_rt + pl.win_tpc);
        p.tile_nt = pl.tile.NT;
        p.seg_len = pl.seg_len;
        p.n_segs = pl.n_segs;
        p.n_ctas = (int64_t)pl.n_nblocks * pl.n_segs * ((n_templates + pl.slide_tpc - 1) / pl.slide_tpc);
        // bounds, pack, window sums (per-tau recurrence / groups of tau: whichever regions exist),
        // slide + closure + marginals, finalize
        p.n_launches = 4 + (pl.mom_n16 > 0) + (pl.grid.N_tau > pl.mom_n16);
    } else if (pl.rect_small) {
        p.kernel = TFSTAT_KERNEL_RECT_SMALL;
        p.tile_c = 1;
        p.tile_nt = 256;
        p.n_ctas = n_templates;
        p.n_launches = 1;
    } else if (pl.rect.enabled) {
        p.kernel = pl.rect.tile ? TFSTAT_KERNEL_RECT_TILE : TFSTAT_KERNEL_RECT_RUN;
        p.tile_c = pl.rect.Q;
        p.tile_nt = rect_run_threads(pl);
        p.seg_len = pl.rect.seg_cols;
        p.n_segs = pl.rect.n_coltiles;
        p.n_ctas = (int64_t)pl.rect.n_rowtiles * pl.rect.n_coltiles * n_templates;
        p.n_launches = 4;  // bounds, prefix + steps, running sums, finalize
    } else {
        p.kernel = TFSTAT_KERNEL_RECT_CELLS;
        p.tile_c = 1;
        p.tile_nt = 256;
        p.n_ctas = (int64_t)pl.cell_blocks_per_template * n_templates;
        p.n_launches = 4;
    }
    const uint32_t n = std::min<uint32_t>(info->struct_size, (uint32_t)sizeof(p));
    p.struct_size = n;
    std::memcpy(info, &p, n);
    return TFSTAT_OK;
}

int tfstat_search(const float *atoms, int64_t template_stride, int64_t ld,
                  const int32_t *t_atoms, int32_t n_atoms, int32_t n_templates, int window,
                  int32_t t0_min, int32_t dt0, int32_t N_t0, int32_t tau_min, int32_t dtau,
                  int32_t N_tau, tfstat_result *out, float *out_maps, uint8_t *out_flags,
                  void *workspace, size_t workspace_bytes, void *stream,
                  const tfstat_opts *opts_host)
{
    if (!atoms || !t_atoms || (!out && !out_maps)) return TFSTAT_EINVAL;
    if (ld < n_atoms || (n_templates > 1 && template_stride < 7 * ld)) return TFSTAT_EINVAL;
    const OptsIn oi(opts_host);
    if (!oi.ok) return TFSTAT_EINVAL;
    const Plan pl = make_plan(window, n_atoms, n_templates, t0_min, dt0, N_t0, tau_min, dtau,
                              N_tau, &oi.o);
    if (pl.status != TFSTAT_OK) return pl.status;
    if (!workspace || workspace_bytes < pl.bytes ||
        (reinterpret_cast<uintptr_t>(workspace) & (kAlign - 1)))
        return TFSTAT_EWORKSPACE;
    return run_device(pl, atoms, template_stride, ld, t_atoms, out, out_maps, out_flags,
                      workspace, static_cast<cudaStream_t>(stream), true);
}

int tfstat_map(const float *atoms, int64_t ld, const int32_t *t_atoms, int32_t n_atoms,
               int window, int32_t t0_min, int32_t dt0, int32_t N_t0, int32_t tau_min,
               int32_t dtau, int32_t N_tau, float *out_map, uint8_t *out_flags,
               void *workspace, size_t workspace_bytes, void *stream,
               const tfstat_opts *opts_host)
{
    if (!out_map) return TFSTAT_EINVAL;
    return tfstat_search(atoms, 7 * ld, ld, t_atoms, n_atoms, 1, window, t0_min, dt0, N_t0,
                         tau_min, dtau, N_tau, nullptr, out_map, out_flags, workspace,
                         workspace_bytes, stream, opts_host);
}

size_t tfstat_marginalise_workspace_bytes(int32_t N_t0, int32_t N_tau)
{
    if (N_t0 < 1 || N_tau < 1) return 0;
    return align_up(sizeof(Partial) * (size_t)marginalise_blocks((int64_t)N_t0 * N_tau));
}

int tfstat_marginalise(const float *map, const uint8_t *flags, int32_t N_t0, int32_t N_tau,
                       tfstat_result *out, void *workspace, size_t workspace_bytes,
                       void *stream, const tfstat_opts *opts_host)
{
    if (!map || !out || N_t0 < 1 || N_tau < 1 || !OptsIn(opts_host).ok) return TFSTAT_EINVAL;
    const int64_t n_cells = (int64_t)N_t0 * N_tau;
    if (n_cells >= (int64_t(1) << 31)) return TFSTAT_EINVAL;
    const int32_t nb = marginalise_blocks(n_cells);
    if (!workspace || workspace_bytes < sizeof(Partial) * (size_t)nb ||
        (reinterpret_cast<uintptr_t>(workspace) & 15u))  // Partial is stored with 16-byte stores
        return TFSTAT_EWORKSPACE;
    TF_CUDA(launch_marginalise(map, flags, n_cells, N_tau, static_cast<Partial *>(workspace),
                               nb, out, static_cast<cudaStream_t>(stream)));
    return TFSTAT_OK;
}

int tfstat_count_terms(const int32_t *t_atoms, int32_t n_atoms, int window, int32_t t0_min,
                       int32_t dt0, int32_t N_t0, int32_t tau_min, int32_t dtau,
                       int32_t N_tau, int64_t *out_terms, void *workspace,
                       size_t workspace_bytes, void *stream, const tfstat_opts *opts_host)
{
    if (!t_atoms || !out_terms || !OptsIn(opts_host).ok) return TFSTAT_EINVAL;
    const Plan pl = make_plan(window, n_atoms, 1, t0_min, dt0, N_t0, tau_min, dtau, N_tau,
                              nullptr);
    if (pl.status != TFSTAT_OK) return pl.status;
    if (!workspace || workspace_bytes < pl.bytes) return TFSTAT_EWORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    TF_CUDA(launch_bounds(pl, t_atoms, workspace, st));
    TF_CUDA(launch_count_terms(pl, make_bounds(pl, t_atoms, workspace), out_terms, st));
    return TFSTAT_OK;
}

int tfstat_validate_timestamps(const int32_t *t_atoms, int32_t n_atoms, int32_t *out_first_bad,
                               void *stream, const tfstat_opts *opts_host)
{
    if (!t_atoms || !out_first_bad || n_atoms < 1 || !OptsIn(opts_host).ok) return TFSTAT_EINVAL;
    TF_CUDA(launch_validate_timestamps(t_atoms, n_atoms, out_first_bad,
                                       static_cast<cudaStream_t>(stream)));
    return TFSTAT_OK;
}

size_t tfstat_general_workspace_bytes(int32_t N_t0, int32_t N_tau)
{
    if (N_t0 < 1 || N_tau < 1 || (int64_t)N_t0 * N_tau >= (int64_t(1) << 31)) return 0;
    return align_up(sizeof(Partial) * (size_t)general_partials(N_t0, N_tau));
}

int tfstat_map_general(const float *atoms, int64_t ld, const int32_t *t_atoms, int32_t n_atoms,
                       const tfstat_window *window_host, const int32_t *t0_grid, int32_t N_t0,
                       const int32_t *tau_grid, int32_t N_tau, float *out_map,
                       uint8_t *out_flags, tfstat_result *out, void *workspace,
                       size_t workspace_bytes, void *stream, const tfstat_opts *opts_host)
{
    if (!atoms || !t_atoms || !window_host || !t0_grid || !tau_grid || (!out_map && !out))
        return TFSTAT_EINVAL;
    const OptsIn oi(opts_host);
    if (!oi.ok) return TFSTAT_EINVAL;
    if (n_atoms < 1 || ld < n_atoms || N_t0 < 1 || N_tau < 1) return TFSTAT_EINVAL;
    if ((int64_t)N_t0 * N_tau >= (int64_t(1) << 31)) return TFSTAT_EINVAL;
    const tfstat_window &w = *window_host;
    if (w.kind != TFSTAT_WINDOW_RECT && w.kind != TFSTAT_WINDOW_EXP &&
        w.kind != TFSTAT_WINDOW_TABLE)
        return TFSTAT_EINVAL;
    if (w.support_num < 1 || w.support_den < 1) return TFSTAT_EINVAL;
    if (w.kind == TFSTAT_WINDOW_TABLE && (!w.table || w.n_table < 2)) return TFSTAT_EINVAL;
    const size_t need = tfstat_general_workspace_bytes(N_t0, N_tau);
    if (!workspace || workspace_bytes < need ||
        (reinterpret_cast<uintptr_t>(workspace) & (kAlign - 1)))
        return TFSTAT_EWORKSPACE;
    const int32_t min_atoms = oi.o.min_atoms > 0 ? oi.o.min_atoms : 2;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    Partial *partials = out ? static_cast<Partial *>(workspace) : nullptr;
    int32_t n_partials = 0;
    TF_CUDA(launch_general(atoms, ld, t_atoms, n_atoms, w, t0_grid, N_t0, tau_grid, N_tau,
                           min_atoms, out_map, out_flags, partials, &n_partials,
                           oi.o.tile_c, st));
    if (out) TF_CUDA(launch_finalize(partials, n_partials, 1, N_tau, out, st));
    return TFSTAT_OK;
}

int tfstat_merge_detectors(const float *const *atoms_dets, const int64_t *template_strides,
                           const int64_t *lds, const int32_t *const *t_dets,
                           const int32_t *n_atoms_dets, int32_t n_det, int32_t n_templates,
                           const int32_t *t_out, int32_t n_out, float *out_atoms,
                           int64_t template_stride_out, int64_t ld_out, void *stream,
                           const tfstat_opts *opts_host)
{
    if (!atoms_dets || !template_strides || !lds || !t_dets || !n_atoms_dets || !t_out ||
        !out_atoms || !OptsIn(opts_host).ok)
        return TFSTAT_EINVAL;
    if (n_det < 1 || n_det > TFSTAT_MAX_DETECTORS || n_templates < 1 || n_out < 1 ||
        ld_out < n_out || (n_templates > 1 && template_stride_out < 7 * ld_out))
        return TFSTAT_EINVAL;
    for (int x = 0; x < n_det; ++x) {
        if (!atoms_dets[x] || !t_dets[x] || n_atoms_dets[x] < 1 || lds[x] < n_atoms_dets[x] ||
            (n_templates > 1 && template_strides[x] < 7 * lds[x]))
            return TFSTAT_EINVAL;
    }
    TF_CUDA(launch_merge(atoms_dets, template_strides, lds, t_dets, n_atoms_dets, n_det,
                         n_templates, t_out, n_out, out_atoms, template_stride_out, ld_out,
                         static_cast<cudaStream_t>(stream)));
    return TFSTAT_OK;
}

int tfstat_search_host(const float *atoms_host, int64_t template_stride, int64_t ld,
                       const int32_t *t_atoms_host, int32_t n_atoms, int32_t n_templates,
                       int window, int32_t t0_min, int32_t dt0, int32_t N_t0, int32_t tau_min,
                       int32_t dtau, int32_t N_tau, tfstat_result *out_host,
                       float *out_maps_host, void *device_scratch, size_t device_scratch_bytes,
                       const tfstat_opts *opts_host)
{
    if (!atoms_host || !t_atoms_host || !out_host) return TFSTAT_EINVAL;
    if (ld < n_atoms || (n_templates > 1 && template_stride < 7 * ld)) return TFSTAT_EINVAL;
    if (n_templates < 1) return TFSTAT_EINVAL;
    const OptsIn oi(opts_host);
    if (!oi.ok) return TFSTAT_EINVAL;
    if (device_scratch && (reinterpret_cast<uintptr_t>(device_scratch) & (kAlign - 1)))
        return TFSTAT_EWORKSPACE;
    const size_t budget = device_scratch_bytes ? device_scratch_bytes : size_t(2) << 30;
    const int64_t cells = (int64_t)N_t0 * N_tau;
    // device layout: two atom buffers (+ two map buffers) of Tc templates, workspace, time
    // stamps, results; Tc = templates per chunk, the largest that fits the budget
    const size_t tpl_bytes = sizeof(float) * (size_t)template_stride;
    const size_t map_bytes = out_maps_host ? sizeof(float) * (size_t)cells : 0;
    const size_t t_bytes = align_up(sizeof(int32_t) * (size_t)n_atoms);
    const size_t out_bytes = align_up(sizeof(tfstat_result) * (size_t)n_templates);
    int32_t Tc = host_chunk_templates(n_templates);
    Plan pl, pl_last;
    size_t need = 0, ws_bytes = 0;
    for (;; Tc = (Tc + 1) / 2) {
        const int st = plan_host_chunks(window, n_atoms, n_templates, Tc, t0_min, dt0, N_t0,
                                        tau_min, dtau, N_tau, &oi.o, pl, pl_last, ws_bytes);
        if (st != TFSTAT_OK) return st;
        need = 2 * (align_up(Tc * tpl_bytes) + align_up(Tc * map_bytes)) + ws_bytes + t_bytes +
               out_bytes;
        if (need <= budget || Tc == 1) break;
    }
    if (device_scratch && need > budget) return TFSTAT_EWORKSPACE;
    const int n_chunks = (n_templates + Tc - 1) / Tc;

    char *base = static_cast<char *>(device_scratch);
    bool own = false;
    cudaStream_t s_copy = nullptr, s_comp = nullptr, s_back = nullptr;
    cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr},
                ev_back[2] = {nullptr, nullptr};
    int rc = TFSTAT_OK;
    auto chk = [&](cudaError_t e) {
        if (e != cudaSuccess && rc == TFSTAT_OK) rc = cuda_fail(e);
        return e == cudaSuccess;
    };
    do {
        if (!base) {
            if (!chk(cudaMalloc(&base, need))) break;
            own = true;
        }
        size_t off = 0;
        auto carve = [&](size_t n) {
            char *q = base + off;
            off += align_up(n);
            return q;
        };
        char *d_atoms[2] = {carve(Tc * tpl_bytes), carve(Tc * tpl_bytes)};
        float *d_maps[2] = {nullptr, nullptr};
        if (map_bytes)
            for (int b = 0; b < 2; ++b) d_maps[b] = reinterpret_cast<float *>(carve(Tc * map_bytes));
        void *d_ws = carve(ws_bytes);
        int32_t *d_t = reinterpret_cast<int32_t *>(carve(sizeof(int32_t) * (size_t)n_atoms));
        tfstat_result *d_out =
            reinterpret_cast<tfstat_result *>(carve(sizeof(tfstat_result) * (size_t)n_templates));

        if (!chk(cudaStreamCreateWithFlags(&s_copy, cudaStreamNonBlocking))) break;
        if (!chk(cudaStreamCreateWithFlags(&s_comp, cudaStreamNonBlocking))) break;
        if (map_bytes && !chk(cudaStreamCreateWithFlags(&s_back, cudaStreamNonBlocking))) break;
        bool ok = true;
        for (int b = 0; b < 2 && ok; ++b) {
            ok = chk(cudaEventCreateWithFlags(&ev_in[b], cudaEventDisableTiming)) &&
                 chk(cudaEventCreateWithFlags(&ev_done[b], cudaEventDisableTiming));
            if (ok && map_bytes)
                ok = chk(cudaEventCreateWithFlags(&ev_back[b], cudaEventDisableTiming));
        }
        if (!ok) break;
        if (!chk(cudaMemcpyAsync(d_t, t_atoms_host, sizeof(int32_t) * (size_t)n_atoms,
                                 cudaMemcpyHostToDevice, s_comp)))
            break;
        // the lo / edge tables depend on the time stamps and the grid only (same offsets in every
        // chunk's plan): built by the first chunk that needs them -- a chunk that takes the
        // one-launch small-map kernel does not, a ragged last chunk after it may
        bool bounds_done = false;
        for (int c = 0; c < n_chunks && rc == TFSTAT_OK; ++c) {
            const int b = c & 1;
            const int32_t k0 = c * Tc;
            const int32_t cnt = std::min<int32_t>(Tc, n_templates - k0);
            const Plan &plc = cnt == Tc ? pl : pl_last;
            // buffer b is free once chunk c-2 has been computed (and its maps copied back)
            if (c >= 2) {
                chk(cudaStreamWaitEvent(s_copy, ev_done[b], 0));
                if (map_bytes) chk(cudaStreamWaitEvent(s_comp, ev_back[b], 0));
            }
            const size_t n_float = (size_t)(cnt - 1) * template_stride + 6 * ld + n_atoms;
            chk(cudaMemcpyAsync(d_atoms[b], atoms_host + (size_t)k0 * template_stride,
                                sizeof(float) * n_float, cudaMemcpyHostToDevice, s_copy));
            chk(cudaEventRecord(ev_in[b], s_copy));
            chk(cudaStreamWaitEvent(s_comp, ev_in[b], 0));
            const bool do_bounds = !bounds_done && !(plc.window == TFSTAT_WINDOW_RECT && plc.rect_small);
            const int r = run_device(plc, reinterpret_cast<const float *>(d_atoms[b]),
                                     template_stride, ld, d_t, d_out + k0, d_maps[b], nullptr,
                                     d_ws, s_comp, do_bounds);
            if (r != TFSTAT_OK) rc = r;
            bounds_done = bounds_done || do_bounds;
            chk(cudaEventRecord(ev_done[b], s_comp));
            if (map_bytes) {
                chk(cudaStreamWaitEvent(s_back, ev_done[b], 0));
                chk(cudaMemcpyAsync(out_maps_host + (size_t)k0 * cells, d_maps[b],
                                    (size_t)cnt * map_bytes, cudaMemcpyDeviceToHost, s_back));
                chk(cudaEventRecord(ev_back[b], s_back));
            }
        }
        if (rc != TFSTAT_OK) break;
        chk(cudaMemcpyAsync(out_host, d_out, sizeof(tfstat_result) * (size_t)n_templates,
                            cudaMemcpyDeviceToHost, s_comp));
    } while (0);
    // (a fault of a kernel or a copy surfaces here: it is this call's error, not a later one's)
    if (s_copy) chk(cudaStreamSynchronize(s_copy));
    if (s_comp) chk(cudaStreamSynchronize(s_comp));
    if (s_back) chk(cudaStreamSynchronize(s_back));
    for (int b = 0; b < 2; ++b) {
        if (ev_in[b]) cudaEventDestroy(ev_in[b]);
        if (ev_done[b]) cudaEventDestroy(ev_done[b]);
        if (ev_back[b]) cudaEventDestroy(ev_back[b]);
    }
    if (s_copy) cudaStreamDestroy(s_copy);
    if (s_comp) cudaStreamDestroy(s_comp);
    if (s_back) cudaStreamDestroy(s_back);
    if (own) cudaFree(base);
    return rc;
}

size_t tfstat_search_host_scratch_bytes(int64_t template_stride, int32_t n_atoms,
                                        int32_t n_templates, int window, int32_t t0_min,
                                        int32_t dt0, int32_t N_t0, int32_t tau_min, int32_t dtau,
                                        int32_t N_tau, int want_maps,
                                        const tfstat_opts *opts_host)
{
    if (n_templates < 1 || template_stride < 1) return 0;
    const OptsIn oi(opts_host);
    if (!oi.ok) return 0;
    const int32_t Tc = host_chunk_templates(n_templates);
    Plan pl, pl_last;
    size_t ws_bytes = 0;
    if (plan_host_chunks(window, n_atoms, n_templates, Tc, t0_min, dt0, N_t0, tau_min, dtau, N_tau,
                         &oi.o, pl, pl_last, ws_bytes) != TFSTAT_OK)
        return 0;
    const size_t tpl_bytes = sizeof(float) * (size_t)template_stride;
    const size_t map_bytes = want_maps ? sizeof(float) * (size_t)N_t0 * N_tau : 0;
    return 2 * (align_up(Tc * tpl_bytes) + align_up(Tc * map_bytes)) + ws_bytes +
           align_up(sizeof(int32_t) * (size_t)n_atoms) +
           align_up(sizeof(tfstat_result) * (size_t)n_templates);
}

}  // extern "C"

// ---------------------------------------------------------------------------------------
// tfstat_marginalise_static: tfstat_marginalise for callers that cannot allocate (code under
// CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc) and have no
// workspace to hand over.  The scratch of the marginalisation -- one Partial per CTA of
// marginalise_kernel, read back by finalize_kernel -- lives in a file-scope __device__ array of
// kStaticPartials records (37 888 bytes; every GPU that loads the library holds it until exit).
// marginalise_blocks() never asks for more than 148 x 8 CTAs, so that serves every map the
// entry point accepts (N_t0 N_tau < 2^31); a request beyond the array is refused.
//
// In host code the array's NAME is a host-side stand-in, not a device address: its address on
// the current device comes from cudaGetSymbolAddress, asked for once per device with that
// device current, and that pointer is what the kernels get.
//
// Every call shares the array.  Nothing in it has to start at zero (every CTA of
// marginalise_kernel writes its own record before finalize_kernel reads any), so a call does
// not care what the last one left; but two calls that OVERLAP on the GPU (different streams,
// or graphs replayed concurrently) race on it.  Calls on one stream are ordered and safe.
// ---------------------------------------------------------------------------------------
namespace {

constexpr int kStaticPartials = 148 * 8;
constexpr int kStaticMaxDevices = 64;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticPartials * sizeof(Partial)];

// device address of g_static_scratch on the CURRENT device; no allocation
int static_scratch(Partial **out)
{
    static std::mutex mu;
    static Partial *ptr[kStaticMaxDevices] = {};
    int dev = -1;
    TF_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return TFSTAT_EINVAL;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        void *p = nullptr;
        TF_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return TFSTAT_EWORKSPACE;
        ptr[dev] = static_cast<Partial *>(p);
    }
    *out = ptr[dev];
    return TFSTAT_OK;
}

}  // namespace

extern "C" {

size_t tfstat_marginalise_static_max_cells(void) { return ((size_t)1 << 31) - 1; }

int tfstat_marginalise_static(const float *map, const uint8_t *flags, int32_t N_t0,
                              int32_t N_tau, tfstat_result *out, void *stream)
{
    if (!map || !out || N_t0 < 1 || N_tau < 1) return TFSTAT_EINVAL;
    const int64_t n_cells = (int64_t)N_t0 * N_tau;
    if ((uint64_t)n_cells > tfstat_marginalise_static_max_cells()) return TFSTAT_EINVAL;
    const int32_t nb = marginalise_blocks(n_cells);
    if (nb > kStaticPartials) return TFSTAT_EWORKSPACE;  // beyond the static scratch
    Partial *scratch = nullptr;
    const int rc = static_scratch(&scratch);
    if (rc != TFSTAT_OK) return rc;
    TF_CUDA(launch_marginalise(map, flags, n_cells, N_tau, scratch, nb, out,
                               static_cast<cudaStream_t>(stream)));
    return TFSTAT_OK;
}

}  // extern "C"
