// sliced_dispatch.cpp - shape table of the bit-sliced kernel instantiations (scan_sliced_inst.cu).
#include "internal.h"

namespace kripke {

typedef int (*sliced_launch_fn)(const ScanJob &, const SlicedPlan &, void *, uint32_t *);

#define SHAPES(X)                                                              \
    X(3, 0, 4) X(4, 0, 4) X(5, 0, 4) X(6, 0, 4)                                \
    X(4, 1, 4) X(5, 1, 4) X(3, 2, 4) X(4, 2, 4)                                \
    X(5, 2, 3) X(5, 2, 4) X(6, 2, 3)                                           \
    X(4, 3, 4) X(5, 3, 3) X(5, 3, 4)

#define DECL(N, K, D) int launch_sliced_##N##_##K##_d##D(const ScanJob &, const SlicedPlan &, void *, uint32_t *);
SHAPES(DECL)
#undef DECL

namespace {
constexpr uint32_t SLICED_MB = 2;   // every instantiation uses M = 4 words per thread
struct Row { uint32_t n, k, dmax; sliced_launch_fn fn; };
#define ROW(N, K, D) {N, K, D, launch_sliced_##N##_##K##_d##D},
const Row kRows[] = {SHAPES(ROW)};
#undef ROW

// the instantiation with the fewest stack slots that still fits `need`
const Row *find(uint32_t n, uint32_t k, uint32_t need) {
    const Row *best = nullptr;
    for (const Row &r : kRows)
        if (r.n == n && r.k == k && r.dmax >= need && (!best || r.dmax < best->dmax)) best = &r;
    return best;
}
}  // namespace

uint64_t sliced_frames_per_unit(uint32_t n, uint32_t k) {
    const uint32_t low = 5 + SLICED_MB;
    return (k * n >= low) ? 1ull : (1ull << (low - k * n));
}

uint32_t sliced_max_need(uint32_t n, uint32_t k, uint32_t cls) {
    // group-per-unit shapes enumerate frames from the model index: class K only
    if (sliced_frames_per_unit(n, k) != 1 && cls != KRIPKE_CLASS_K) return 0;
    uint32_t m = 0;
    for (const Row &r : kRows)
        if (r.n == n && r.k == k && r.dmax > m) m = r.dmax;
    return m;
}

int launch_sliced(const ScanJob &job, const SlicedPlan &plan, void *stream, uint32_t *launches) {
    const Row *r = find(job.n, job.k, plan.max_need);
    if (!r) return 801;   // cudaErrorNotSupported
    return r->fn(job, plan, stream, launches);
}

}  // namespace kripke
