// general.cu -- tfstat_map_general: the map for a general window function on explicit
// (possibly irregular) t0 / tau arrays (R17).
//
// "Different window functions for the amplitude evolution could also be considered, and would
// generically follow the GPU kernel grid setup and timing model for the exponential window,
// since it does not assume any function-specific optimisations"; the grid may
// have "a coarser or even variable sampling".  So this is the direct truncated
// sum per cell, with
//   membership  t0 <= t_a  and  (t_a - t0) * den < num * tau        (integers, half-open)
//   weight      w(u), u = (t_a - t0) / tau:  1 | exp(-u) | linear interpolation of a table
//   w on Fa, Fb and w^2 on a2, b2, ab; closure eq. (7); marginals eq. (5).
//
// One thread owns one cell at a time: a CTA is (one t0) x (NT consecutive entries of the tau
// array).  Window bounds come from two binary searches per cell (no lattice: the arrays are
// arbitrary).  The CTA streams the atoms [lo, max hi) through shared memory in chunks, staged
// once as (dt, ab | a2, b2) and (Re Fa, Im Fa | Re Fb, Im Fb) records that every lane reads by
// broadcast; each thread stops at its own hi.  No weight sharing between cells is assumed (a
// general w(u) does not factorise), so the executed mix is the algorithmic one: per term the
// weight, w^2, and 7 fp32 multiply-adds (4 packed fma.rn.f32x2).  The closure runs in fp64.
#include "plan.h"

// unroll of the atom loop: swept 2..32 on B200, 16 is 4-5 % faster than 4
constexpr int kAtomUnroll = 16;
namespace tfstat {

namespace {

constexpr int kGenNT = 128;
constexpr int kGenKC = 512;        // atoms per staged chunk (16 KB)
constexpr int kGenTableSmem = 4096;  // tables up to this many samples are staged in smem

struct GeneralArgs {
    const float *atoms;
    int64_t ld;
    const int32_t *t;
    int32_t n_atoms;
    const int32_t *t0_grid;
    int32_t N_t0;
    const int32_t *tau_grid;
    int32_t N_tau;
    int32_t sup_num, sup_den;
    const float *table;
    int32_t n_table;
    int32_t min_atoms;
    float *out_map;
    uint8_t *out_flags;
};

// fp64 redo of a short, ill-conditioned window (tfstat_dev.cuh, closure_2F_exp): the window's
// sums straight from the atoms with the weight of the kind evaluated in fp64
template <int KIND>
__device__ __noinline__ Sums64 general_resum64(const GeneralArgs &a, const int lo, const int hi,
                                               const long long t0, const double tau)
{
    Sums64 s;
    s.A = s.B = s.C = s.far = s.fai = s.fbr = s.fbi = 0.0;
    const double support = (double)a.sup_num / (double)a.sup_den;
    for (int al = lo; al < hi; ++al) {
        const double u = (double)((long long)__ldg(a.t + al) - t0) / tau;
        double w = 1.0;
        if (KIND == TFSTAT_WINDOW_EXP) {
            w = exp(-u);
        } else if (KIND == TFSTAT_WINDOW_TABLE) {
            const double x = u / support * (double)(a.n_table - 1);
            int k = (int)floor(x);
            k = max(0, min(k, a.n_table - 2));
            const double t0v = (double)__ldg(a.table + k), t1v = (double)__ldg(a.table + k + 1);
            w = t0v + (x - (double)k) * (t1v - t0v);
        }
        const double w2 = w * w;
        s.A += w2 * (double)__ldg(a.atoms + al);
        s.B += w2 * (double)__ldg(a.atoms + a.ld + al);
        s.C += w2 * (double)__ldg(a.atoms + 2 * a.ld + al);
        s.far += w * (double)__ldg(a.atoms + 3 * a.ld + al);
        s.fai += w * (double)__ldg(a.atoms + 4 * a.ld + al);
        s.fbr += w * (double)__ldg(a.atoms + 5 * a.ld + al);
        s.fbi += w * (double)__ldg(a.atoms + 6 * a.ld + al);
    }
    return s;
}

// CT cells per thread (consecutive tau indices of the CTA's NT x CT block): one broadcast read
// of an atom record serves CT cells; the weights stay per cell.  With CT = 1 the two LDS.128 per
// term put the L1 wavefront counter at 78 % of its peak (ncu), but measured on B200 CT = 2 is
// only 3 % faster (configs 2, 3, 5) and CT = 4 is 7-20 % slower (fewer, longer CTAs; one select
// per term for the ragged window ends): the kernel is bound by its ~11 instructions per term.
template <int KIND, int CT>
__global__ void __launch_bounds__(kGenNT)
    general_kernel(const GeneralArgs a, Partial *__restrict__ partials, const int n_nblocks)
{
    __shared__ ulonglong2 s_a[kGenKC];
    __shared__ ulonglong2 s_b[kGenKC];
    __shared__ Marg s_red[32];
    __shared__ int s_hi[kGenNT / 32];
    __shared__ float s_tab[KIND == TFSTAT_WINDOW_TABLE ? kGenTableSmem : 1];

    const int m = blockIdx.x / n_nblocks;
    // a thread's CT cells are CONSECUTIVE entries of the tau array: on a sorted array their
    // windows have nearly the same length, so little of the shared atom loop is wasted
    const int n0 = (blockIdx.x % n_nblocks) * (kGenNT * CT) + threadIdx.x * CT;
    const long long t0 = __ldg(a.t0_grid + m);
    // a1: bounds.  dt * den < num * tau  <=>  t < t0 + ceil(num tau / den)
    const int lo = lower_bound_t(a.t, a.n_atoms, t0);
    long long tau[CT];
    int hi[CT];
    float kw[CT];  // exp: w = 2^(dt * kw); table: x = dt * kw, knots at integer x
    int hmax = lo;
#pragma unroll
    for (int c = 0; c < CT; ++c) {
        const int n = n0 + c;
        tau[c] = n < a.N_tau ? (long long)__ldg(a.tau_grid + n) : 0;
        hi[c] = lo;
        kw[c] = 0.0f;
        if (tau[c] >= 1) {
            const long long len = ((long long)a.sup_num * tau[c] + a.sup_den - 1) / a.sup_den;
            hi[c] = lower_bound_t(a.t, a.n_atoms, t0 + len);
            kw[c] = KIND == TFSTAT_WINDOW_EXP
                        ? (float)(-1.4426950408889634 / (double)tau[c])
                        : (float)((double)(a.n_table - 1) * (double)a.sup_den /
                                  ((double)a.sup_num * (double)tau[c]));
        }
        hmax = max(hmax, hi[c]);
    }
    // atom range of the CTA: [lo, max over its cells of hi)
    const int my_e = hmax;
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) hmax = max(hmax, __shfl_xor_sync(0xffffffffu, hmax, s));
    if ((threadIdx.x & 31) == 0) s_hi[threadIdx.x >> 5] = hmax;
    const bool tab_smem = KIND == TFSTAT_WINDOW_TABLE && a.n_table <= kGenTableSmem;
    if (tab_smem)
        for (int i = threadIdx.x; i < a.n_table; i += kGenNT) s_tab[i] = __ldg(a.table + i);
    __syncthreads();
    int cta_e = s_hi[0];
#pragma unroll
    for (int w = 1; w < kGenNT / 32; ++w) cta_e = max(cta_e, s_hi[w]);
    const float *__restrict__ tab = tab_smem ? s_tab : a.table;

    u64 acc_ab[CT], acc_fa[CT], acc_fb[CT];  // (A, B), (Re Fa, Im Fa), (Re Fb, Im Fb)
    float acc_c[CT];
#pragma unroll
    for (int c = 0; c < CT; ++c) {
        acc_ab[c] = acc_fa[c] = acc_fb[c] = 0ull;
        acc_c[c] = 0.0f;
    }
#pragma unroll 1
    for (int cs = lo; cs < cta_e; cs += kGenKC) {
        const int n_stage = min(kGenKC, cta_e - cs);
        for (int i = threadIdx.x; i < n_stage; i += kGenNT) {  // a0: stage atoms [cs, cs+n_stage)
            const int al = cs + i;
            const float dt = (float)((long long)__ldg(a.t + al) - t0);
            ulonglong2 ra, rb;
            ra.x = pack2(dt, __ldg(a.atoms + 2 * a.ld + al));
            ra.y = pack2(__ldg(a.atoms + al), __ldg(a.atoms + a.ld + al));
            rb.x = pack2(__ldg(a.atoms + 3 * a.ld + al), __ldg(a.atoms + 4 * a.ld + al));
            rb.y = pack2(__ldg(a.atoms + 5 * a.ld + al), __ldg(a.atoms + 6 * a.ld + al));
            s_a[i] = ra;
            s_b[i] = rb;
        }
        __syncthreads();
        const int x1 = min(cs + n_stage, my_e) - cs;  // this thread's atoms of the chunk: [0, x1)
#pragma unroll kAtomUnroll
        for (int i = 0; i < x1; ++i) {
            const ulonglong2 ra = s_a[i], rb = s_b[i];
            float dt, ab;
            unpack2(ra.x, dt, ab);
#pragma unroll
            for (int c = 0; c < CT; ++c) {
                float w;
                if (KIND == TFSTAT_WINDOW_RECT) {
                    w = 1.0f;
                } else if (KIND == TFSTAT_WINDOW_EXP) {
                    w = ex2_approx(dt * kw[c]);
                } else {
                    const float x = dt * kw[c];
                    const int k = min((int)x, a.n_table - 2);
                    const float t0v = tab[k], t1v = tab[k + 1];
                    w = fmaf(x - (float)k, t1v - t0v, t0v);
                }
                // an atom beyond this cell's own window is SKIPPED, not weighted by zero: 0 x NaN of
                // a non-finite atom (a bad SFT) would spoil windows it is not part of
                if (CT == 1 || cs + i < hi[c]) {
                    const float w2 = w * w;
                    ffma2(acc_ab[c], pack2(w2, w2), ra.y);
                    const u64 ww = pack2(w, w);
                    ffma2(acc_fa[c], ww, rb.x);
                    ffma2(acc_fb[c], ww, rb.y);
                    acc_c[c] = fmaf(w2, ab, acc_c[c]);
                }
            }
        }
        __syncthreads();
    }

    // a4 closure + a5 marginals
    Marg mg;
    marg_init(mg);
#pragma unroll
    for (int c = 0; c < CT; ++c) {
        const int n = n0 + c;
        if (n >= a.N_tau) continue;
        Sums64 s;
        float A, B, far, fai, fbr, fbi;
        unpack2(acc_ab[c], A, B);
        unpack2(acc_fa[c], far, fai);
        unpack2(acc_fb[c], fbr, fbi);
        s.A = A;
        s.B = B;
        s.C = acc_c[c];
        s.far = far;
        s.fai = fai;
        s.fbr = fbr;
        s.fbi = fbi;
        const int cnt = hi[c] - lo;
        if (cnt >= 1 && cnt <= kRedoMaxAtoms &&
            !(s.A * s.B - s.C * s.C > 0.015625 * s.A * s.B))
            s = general_resum64<KIND>(a, lo, hi[c], t0, (double)tau[c]);
        uint32_t fl;
        const float twoF = closure_2F(s, cnt, a.min_atoms, fl);
        const int32_t flat = m * a.N_tau + n;
        if (a.out_map) a.out_map[flat] = twoF;
        if (a.out_flags) a.out_flags[flat] = (uint8_t)fl;
        if (!fl) marg_add(mg, twoF, flat);
    }
    if (partials) {
        marg_block_reduce<kGenNT>(mg, s_red);
        if (threadIdx.x == 0) partial_store(partials + blockIdx.x, mg);
    }
}

template <int KIND>
cudaError_t launch_kind(const GeneralArgs &a, Partial *partials, int ct, cudaStream_t st)
{
    const int n_nblocks = (a.N_tau + kGenNT * ct - 1) / (kGenNT * ct);
    const unsigned grid = (unsigned)a.N_t0 * (unsigned)n_nblocks;
    switch (ct) {
    case 4: general_kernel<KIND, 4><<<grid, kGenNT, 0, st>>>(a, partials, n_nblocks); break;
    case 2: general_kernel<KIND, 2><<<grid, kGenNT, 0, st>>>(a, partials, n_nblocks); break;
    default: general_kernel<KIND, 1><<<grid, kGenNT, 0, st>>>(a, partials, n_nblocks); break;
    }
    return cudaGetLastError();
}

}  // namespace

int32_t general_partials(int32_t N_t0, int32_t N_tau)
{
    return N_t0 * ((N_tau + kGenNT - 1) / kGenNT);
}

cudaError_t launch_general(const float *atoms, int64_t ld, const int32_t *t_atoms, int32_t n_atoms,
                           const tfstat_window &w, const int32_t *t0_grid, int32_t N_t0,
                           const int32_t *tau_grid, int32_t N_tau, int32_t min_atoms,
                           float *out_map, uint8_t *out_flags, Partial *partials,
                           int32_t *n_partials, int32_t ct_override, cudaStream_t st)
{
    GeneralArgs a;
    a.atoms = atoms;
    a.ld = ld;
    a.t = t_atoms;
    a.n_atoms = n_atoms;
    a.t0_grid = t0_grid;
    a.N_t0 = N_t0;
    a.tau_grid = tau_grid;
    a.N_tau = N_tau;
    a.sup_num = w.support_num;
    a.sup_den = w.support_den;
    a.table = w.table;
    a.n_table = w.n_table;
    a.min_atoms = min_atoms;
    a.out_map = out_map;
    a.out_flags = out_flags;
    // cells per thread: 2 while that still leaves ~8 CTAs per SM, else 1 (4 only on request)
    auto ctas = [&](int ct) { return (int64_t)N_t0 * ((N_tau + kGenNT * ct - 1) / (kGenNT * ct)); };
    int ct = (N_tau >= 2 * kGenNT && ctas(2) >= 148 * 8) ? 2 : 1;
    if (ct_override == 1 || ct_override == 2 || ct_override == 4) ct = ct_override;
    *n_partials = (int32_t)ctas(ct);
    switch (w.kind) {
    case TFSTAT_WINDOW_RECT: return launch_kind<TFSTAT_WINDOW_RECT>(a, partials, ct, st);
    case TFSTAT_WINDOW_EXP: return launch_kind<TFSTAT_WINDOW_EXP>(a, partials, ct, st);
    case TFSTAT_WINDOW_TABLE: return launch_kind<TFSTAT_WINDOW_TABLE>(a, partials, ct, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace tfstat
