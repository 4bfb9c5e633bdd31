// merge.cu -- tfstat_merge_detectors: per-detector atoms -> atoms merged per time stamp
// (R18).  The paper's atoms carry an index "over SFTs"
// (PAPER.md:65); the map entry points take them merged per time stamp, and this is the merge:
//   out[k][ch][i] = sum over detectors X (in the order given) of atoms_X[k][ch][j], t_X[j] == t_out[i]
// in fp32, fixed order, so the result is reproducible to the bit.  One thread per output time
// stamp finds its atom in every detector by binary search (time stamps are shared by all
// templates, so the search is done once per CTA row and reused for the blockIdx.y templates).
#include <algorithm>

#include "plan.h"

namespace tfstat {

namespace {

constexpr int kMergeNT = 128;
constexpr int kMergeRows = 48;  // grid.y: a thread amortises its binary searches over T / 48 templates

struct MergeArgs {
    const float *atoms[TFSTAT_MAX_DETECTORS];
    const int32_t *t[TFSTAT_MAX_DETECTORS];
    int64_t tstride[TFSTAT_MAX_DETECTORS];
    int64_t ld[TFSTAT_MAX_DETECTORS];
    int32_t n[TFSTAT_MAX_DETECTORS];
    int32_t n_det;
    const int32_t *t_out;
    int32_t n_out;
    int32_t n_templates;
    float *out;
    int64_t tstride_out, ld_out;
};

__global__ void __launch_bounds__(kMergeNT) merge_kernel(const MergeArgs a)
{
    const int i = blockIdx.x * kMergeNT + threadIdx.x;
    if (i >= a.n_out) return;
    const long long ti = __ldg(a.t_out + i);
    int j[TFSTAT_MAX_DETECTORS];
#pragma unroll
    for (int x = 0; x < TFSTAT_MAX_DETECTORS; ++x) {
        j[x] = -1;
        if (x < a.n_det) {
            const int p = lower_bound_t(a.t[x], a.n[x], ti);
            if (p < a.n[x] && (long long)__ldg(a.t[x] + p) == ti) j[x] = p;
        }
    }
    for (int k = blockIdx.y; k < a.n_templates; k += gridDim.y) {
        float acc[7] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
        for (int x = 0; x < TFSTAT_MAX_DETECTORS; ++x) {
            if (j[x] < 0) continue;
            const float *__restrict__ src = a.atoms[x] + (int64_t)k * a.tstride[x] + j[x];
#pragma unroll
            for (int ch = 0; ch < 7; ++ch) acc[ch] += __ldg(src + ch * a.ld[x]);
        }
        float *__restrict__ dst = a.out + (int64_t)k * a.tstride_out + i;
#pragma unroll
        for (int ch = 0; ch < 7; ++ch) dst[ch * a.ld_out] = acc[ch];
    }
}

}  // namespace

cudaError_t launch_merge(const float *const *atoms, const int64_t *tstrides, const int64_t *lds,
                         const int32_t *const *ts, const int32_t *ns, int32_t n_det,
                         int32_t n_templates, const int32_t *t_out, int32_t n_out, float *out,
                         int64_t tstride_out, int64_t ld_out, cudaStream_t st)
{
    MergeArgs a;
    for (int x = 0; x < TFSTAT_MAX_DETECTORS; ++x) {
        a.atoms[x] = x < n_det ? atoms[x] : nullptr;
        a.t[x] = x < n_det ? ts[x] : nullptr;
        a.tstride[x] = x < n_det ? tstrides[x] : 0;
        a.ld[x] = x < n_det ? lds[x] : 0;
        a.n[x] = x < n_det ? ns[x] : 0;
    }
    a.n_det = n_det;
    a.t_out = t_out;
    a.n_out = n_out;
    a.n_templates = n_templates;
    a.out = out;
    a.tstride_out = tstride_out;
    a.ld_out = ld_out;
    const dim3 grid((unsigned)((n_out + kMergeNT - 1) / kMergeNT),
                    (unsigned)std::min<int32_t>(n_templates, kMergeRows), 1);
    merge_kernel<<<grid, kMergeNT, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace tfstat
