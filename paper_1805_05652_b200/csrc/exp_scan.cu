// exp_scan.cu -- exact factorised exponential-window path (SURVEY.md 8(a) row a3').
// Not implemented yet: the plan rejects nothing, the launcher reports it.
#include "plan.h"

namespace tfstat {

cudaError_t launch_exp_scan(const Plan &, const Problem &, float *, Partial *, cudaStream_t)
{
    return cudaErrorNotSupported;
}

}  // namespace tfstat
