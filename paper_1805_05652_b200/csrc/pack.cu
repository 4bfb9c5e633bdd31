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
// the same instruction count as the multiply it replaces.
#include "plan.h"

namespace tfstat {

namespace {

constexpr int kPackNT = 256;

__global__ void __launch_bounds__(kPackNT)
    pack_atoms_kernel(const float *__restrict__ atoms, const int64_t template_stride,
                      const int64_t ld, const int32_t *__restrict__ t, const int n_atoms,
                      const int n_pad, ulonglong2 *__restrict__ rec)
{
    pdl_trigger();
    const int i = blockIdx.x * kPackNT + threadIdx.x;
    const int tpl = blockIdx.y;
    if (i < n_pad) {
        ulonglong2 ra = make_ulonglong2(0ull, 0ull), rb = ra;  // padding: zeros, never summed
        if (i < n_atoms) {
            const float *__restrict__ base = atoms + (int64_t)tpl * template_stride + i;
            const float dtc = (float)((long long)__ldg(t + i) - (long long)__ldg(t + i - i % kPackBlock));
            ra.x = pack2(dtc, __ldg(base + 2 * ld));
            ra.y = pack2(__ldg(base), __ldg(base + ld));
            rb.x = pack2(__ldg(base + 3 * ld), __ldg(base + 4 * ld));
            rb.y = pack2(__ldg(base + 5 * ld), __ldg(base + 6 * ld));
        }
        ulonglong2 *__restrict__ dst = rec + ((int64_t)tpl * n_pad + i) * 2;
        dst[0] = ra;
        dst[1] = rb;
    }
    // nothing here depends on the kernel in front (bounds), but the kernel BEHIND this one
    // relies on "my predecessor is complete => everything before it is too"
    pdl_wait();
}

}  // namespace

cudaError_t launch_pack(const Plan &pl, const Problem &pr, void *packed, cudaStream_t st)
{
    const dim3 grid((unsigned)((pl.n_pad + kPackNT - 1) / kPackNT), (unsigned)pl.n_templates, 1);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(kPackNT, 1, 1);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, pack_atoms_kernel, pr.atoms, pr.template_stride, pr.ld,
                              pr.bounds.t, pl.n_atoms, pl.n_pad,
                              static_cast<ulonglong2 *>(packed));
}

}  // namespace tfstat
