// pack.cu -- step a0 for the exponential-window kernels: the caller's atoms (7 SoA rows of fp32
// + shared int32 time stamps) are packed ONCE per call into 32-byte records
//     rec[2 i]     = { dtc_i, ab_i | a2_i, b2_i }          (the order the kernels consume them in)
//     rec[2 i + 1] = { Re Fa_i, Im Fa_i | Re Fb_i, Im Fb_i }
// so that a kernel can stage a run of atoms with ONE bulk asynchronous copy (cp.async.bulk,
// the 1-D TMA path: no thread touches the data on its way to shared memory) and fetch a single
// atom with two 16-byte loads instead of eight scalar ones.
//
// dtc_i = (float)(t_i - t_{block(i)}), block(i) = i - i % kPackBlock: the time stamp relative to the
// first atom of its block of kPackBlock atoms, exact in fp32 while a block spans < 2^24 s (194
// days).  A kernel turns it into its own weight argument with one FMA:
//     (t_i - t_ref) k = dtc_i k + c,   c = (t_{block(i)} - t_ref) k   (per thread and block),
// the same instruction count as the multiply it replaces.  Atoms that are not finite become
// dtc = NaN with zero channels, and the SIGN bit of dtc marks the atoms at which the time step
// changes (see below): readers take |dtc|.
#include "plan.h"

namespace tfstat {

namespace {

constexpr int kPackNT = 256;

__global__ void __launch_bounds__(kPackNT)
    pack_atoms_kernel(const float *__restrict__ atoms, const int64_t template_stride,
                      const int64_t ld, const int32_t *__restrict__ t, const int n_atoms,
                      const int n_pad, ulonglong2 *__restrict__ rec)
{
    const int i = blockIdx.x * kPackNT + threadIdx.x;
    const int tpl = blockIdx.y;
    if (i < n_pad) {
        ulonglong2 ra = make_ulonglong2(0ull, 0ull), rb = ra;  // padding: zeros, never summed
        if (i < n_atoms) {
            const float *__restrict__ base = atoms + (int64_t)tpl * template_stride + i;
            const long long ti = __ldg(t + i);
            float dtc = (float)(ti - (long long)__ldg(t + i - i % kPackBlock));
            float x[7];
            bool bad = false;
#pragma unroll
            for (int k = 0; k < 7; ++k) {
                x[k] = __ldg(base + k * ld);
                bad = bad || !(fabsf(x[k]) < INFINITY);
            }
            // An atom that is not finite (a bad SFT) is stored as dtc = NaN with zero channels:
            // its WEIGHT is then NaN in every window that holds it (those cells are flagged
            // D <= 0, as in the oracle), while a kernel that masks atoms outside a window with a
            // zero weight gets 0 x 0 = 0 there, not 0 x NaN.
            if (bad) {
                dtc = nanf("");
#pragma unroll
                for (int k = 0; k < 7; ++k) x[k] = 0.0f;
            }
            // Sign bit of dtc: "the step t_{i+1} - t_i differs from the step behind it" (or there
            // is none, or this atom is a bad one).  exp_window_kernel walks the atoms backwards
            // with the multiplicative recurrence S_i = x_i + f S_{i+1}, f = exp(-(t_{i+1} - t_i)/tau):
            // f only has to be recomputed where this bit is set, i.e. at the edges of gaps.
            bool change = i + 2 >= n_atoms || bad;
            if (!change) {
                const long long t1 = __ldg(t + i + 1), t2 = __ldg(t + i + 2);
                change = (t1 - ti) != (t2 - t1);
            }
            // (assembled as integers: a NaN moved through float arithmetic may lose its sign bit)
            unsigned dtc_bits = bad ? 0x7fc00000u : __float_as_uint(dtc);
            if (change) dtc_bits |= 0x80000000u;
            ra.x = ((u64)__float_as_uint(x[2]) << 32) | (u64)dtc_bits;
            ra.y = pack2(x[0], x[1]);
            rb.x = pack2(x[3], x[4]);
            rb.y = pack2(x[5], x[6]);
        }
        ulonglong2 *__restrict__ dst = rec + ((int64_t)tpl * n_pad + i) * 2;
        dst[0] = ra;
        dst[1] = rb;
    }
}

}  // namespace

cudaError_t launch_pack(const Plan &pl, const Problem &pr, void *packed, cudaStream_t st)
{
    const dim3 grid((unsigned)((pl.n_pad + kPackNT - 1) / kPackNT), (unsigned)pl.n_templates, 1);
    pack_atoms_kernel<<<grid, kPackNT, 0, st>>>(pr.atoms, pr.template_stride, pr.ld, pr.bounds.t,
                                                pl.n_atoms, pl.n_pad,
                                                static_cast<ulonglong2 *>(packed));
    return cudaGetLastError();
}

}  // namespace tfstat
