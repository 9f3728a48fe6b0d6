// scan_sliced_inst.cu - explicit instantiations of the bit-sliced kernel, compiled once per
// KRIPKE_INST_GROUP so the groups build in parallel.  INST(n, k, MB, DMAX, TPB, MINB): M = 2^MB
// words per thread, DMAX register-stack slots, TPB threads per block, MINB = minimum resident blocks
// per SM (register budget per thread = 65536 / (TPB * MINB)).  Keep in step with sliced_dispatch.cpp.
#include "scan_sliced.cuh"

#ifndef KRIPKE_INST_GROUP
#error "compile with -DKRIPKE_INST_GROUP=<0..3>"
#endif

namespace kripke {

#define INST(N, K, MB, DMAX, TPB, MINB)                                                             \
    int launch_sliced_##N##_##K##_m##MB##_d##DMAX(const ScanJob &j, const SlicedPlan &p, void *s,    \
                                                  uint32_t *l) {                                     \
        return launch_sliced_inst<SlicedCfg<N, K, MB, DMAX>, TPB, MINB>(j, p, s, l);                \
    }

#if KRIPKE_INST_GROUP == 0
INST(3, 0, 2, 4, 256, 2) INST(4, 0, 2, 4, 256, 2) INST(5, 0, 2, 2, 128, 4) INST(5, 0, 2, 4, 128, 3) INST(6, 0, 2, 2, 128, 3) INST(6, 0, 2, 4, 128, 2)
#elif KRIPKE_INST_GROUP == 1
INST(4, 1, 2, 4, 256, 2) INST(5, 1, 2, 4, 128, 3) INST(5, 1, 4, 1, 128, 3) INST(5, 1, 0, 4, 128, 4) INST(3, 2, 2, 4, 256, 2) INST(4, 2, 3, 2, 128, 3) INST(4, 2, 2, 4, 128, 3)
#elif KRIPKE_INST_GROUP == 2
INST(5, 2, 4, 1, 128, 3) INST(5, 2, 3, 1, 128, 4) INST(5, 2, 3, 2, 128, 3) INST(5, 2, 4, 2, 128, 2) INST(5, 2, 2, 3, 128, 3) INST(5, 2, 2, 4, 128, 2) INST(6, 2, 2, 3, 128, 2)
#elif KRIPKE_INST_GROUP == 3
INST(4, 3, 2, 4, 128, 2) INST(5, 3, 3, 2, 128, 2) INST(5, 3, 2, 3, 128, 2) INST(5, 3, 2, 4, 128, 2)
#endif

}  // namespace kripke
