// sliced_dispatch.cpp - shape table of the bit-sliced kernel instantiations (scan_sliced_inst.cu).
#include "internal.h"

namespace kripke {

typedef int (*sliced_launch_fn)(const ScanJob &, const SlicedPlan &, void *, uint32_t *);

// X(n, k, MB, DMAX)
#define SHAPES(X) \
    X(3, 0, 2, 4) X(4, 0, 2, 4) X(5, 0, 2, 2) X(5, 0, 2, 4) X(6, 0, 2, 2) \
    X(6, 0, 2, 4) X(4, 1, 2, 4) X(5, 1, 2, 4) X(5, 1, 4, 1) X(5, 1, 0, 4) X(3, 2, 2, 4) X(4, 2, 3, 2) \
    X(4, 2, 2, 4) X(5, 2, 4, 1) X(5, 2, 3, 1) X(5, 2, 3, 2) X(5, 2, 4, 2) X(5, 2, 2, 3) X(5, 2, 2, 4) \
    X(6, 2, 2, 3) X(4, 3, 2, 4) X(5, 3, 3, 2) X(5, 3, 2, 3) X(5, 3, 2, 4)

#define DECL(N, K, MB, D) \
    int launch_sliced_##N##_##K##_m##MB##_d##D(const ScanJob &, const SlicedPlan &, void *, uint32_t *);
SHAPES(DECL)
#undef DECL

namespace {
struct Row { uint32_t n, k, mb, dmax; sliced_launch_fn fn; };
#define ROW(N, K, MB, D) {N, K, MB, D, launch_sliced_##N##_##K##_m##MB##_d##D},
const Row kRows[] = {SHAPES(ROW)};
#undef ROW

bool frame_per_unit(const Row &r) { return r.k * r.n >= 5 + r.mb; }

// The instantiation with the fewest stack slots that still fits `need`; among those the one with
// the most words per thread.
const Row *find(uint32_t n, uint32_t k, uint32_t cls, uint32_t need) {
    const Row *best = nullptr;
    for (const Row &r : kRows) {
        if (r.n != n || r.k != k || r.dmax < need) continue;
        // group-per-unit shapes enumerate frames from the model index: class K only
        if (!frame_per_unit(r) && cls != KRIPKE_CLASS_K) continue;
        if (!best || r.dmax < best->dmax || (r.dmax == best->dmax && r.mb > best->mb)) best = &r;
    }
    return best;
}
}  // namespace

bool sliced_select(uint32_t n, uint32_t k, uint32_t cls, uint32_t need, uint64_t *frames_per_unit) {
    const Row *r = find(n, k, cls, need);
    if (!r) return false;
    if (frames_per_unit) *frames_per_unit = frame_per_unit(*r) ? 1ull : (1ull << (5 + r->mb - r->k * r->n));
    return true;
}

uint32_t sliced_row(uint32_t n, uint32_t k, uint32_t cls, uint32_t need) {
    const Row *r = find(n, k, cls, need);
    return r ? (uint32_t)(r - kRows) : UINT32_MAX;
}

uint32_t sliced_lower_mode(uint32_t n, uint32_t k, uint32_t cls) {
    const uint32_t fuse = LOWER_FUSE;
    // every row of one (n, k) that a class can use has the same layout kind (see SHAPES above)
    const Row *r = find(n, k, cls, 1);
    if (!r) return 0;
    return fuse | LOWER_LEAF_DEAD | ((frame_per_unit(*r) && k >= 1 && n <= 5) ? LOWER_LEAF_P : 0u);
}

// Fused micro-ops (LOWER_FUSE) pay off on the one-slot instantiations only: programs
// whose need class runs on a kernel with more slots are lowered without them.
bool sliced_fuses(uint32_t n, uint32_t k, uint32_t need) {
    const Row *r = find(n, k, KRIPKE_CLASS_K, need);
    return r && r->dmax == 1;
}

int launch_sliced(const ScanJob &job, const SlicedPlan &plan, void *stream, uint32_t *launches) {
    // group-per-unit shapes need the range aligned to the unit of the row (the caller aligns to the
    // largest unit of the rows it uses)
    const Row *r = find(job.n, job.k, job.cls, plan.max_need);
    if (!r) return 801;   // cudaErrorNotSupported
    return r->fn(job, plan, stream, launches);
}

}  // namespace kripke
