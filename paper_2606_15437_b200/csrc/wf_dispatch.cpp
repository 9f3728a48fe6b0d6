// wf_dispatch.cpp - table of the warp-frame kernel instantiations (scan_wf_inst.cu).
#include <cuda_runtime.h>

#include "internal.h"

namespace kripke {

extern const WfRow kWfRow0, kWfRow1, kWfRow2, kWfRow3, kWfRow4;

namespace {
const WfRow *const kWfRows[] = {&kWfRow0, &kWfRow1, &kWfRow2, &kWfRow3, &kWfRow4};

const WfRow *wf_find(uint32_t n, uint32_t k, uint32_t cls) {
    for (const WfRow *r : kWfRows)
        if (r->n == n && r->k == k && r->cls == cls) return r;
    return nullptr;
}
}  // namespace

bool wf_select(uint32_t n, uint32_t k, uint32_t cls, uint64_t *frames_per_unit) {
    const WfRow *r = wf_find(n, k, cls);
    if (!r) return false;
    if (frames_per_unit) *frames_per_unit = r->frames_per_unit;
    return true;
}

int launch_wf(const ScanJob &job, const WfPlan &plan, void *stream, uint32_t *launches) {
    const WfRow *r = wf_find(job.n, job.k, job.cls);
    if (!r) return (int)cudaErrorNotSupported;
    return r->launch(job, plan, stream, launches);
}

double wf_cost_per_frame(uint32_t n, uint32_t k, uint32_t cls, const WfOpCounts &c) {
    const WfRow *r = wf_find(n, k, cls);
    return r ? r->cost(c) : 0.0;
}

}  // namespace kripke
