// scan_frames_inst.cu - explicit instantiations of the frame-list kernel (scan_frames.cuh), compiled
// once per KRIPKE_FR_GROUP so the groups build in parallel.  N worlds x VB valuations per pass.
#include "scan_frames.cuh"

#ifndef KRIPKE_FR_GROUP
#error "compile with -DKRIPKE_FR_GROUP=<0..3>"
#endif

namespace kripke {

#define FR_INST(N, VB)                                                                                   \
    int launch_frames_##N##_v##VB(const FramesJob &j, const SlicedPlan &p, void *s, uint32_t *l) {       \
        return launch_frames_inst<N, VB>(j, p, s, l);                                                    \
    }
// VB = 4 is used for n <= 12 only (scan_frames.cu); the larger sizes alias VB = 2
#define FR_ALIAS4(N)                                                                                     \
    int launch_frames_##N##_v4(const FramesJob &j, const SlicedPlan &p, void *s, uint32_t *l) {          \
        return launch_frames_inst<N, 2>(j, p, s, l);                                                     \
    }
#define FR_ALL(N) FR_INST(N, 1) FR_INST(N, 2) FR_INST(N, 4)
#define FR_BIG(N) FR_INST(N, 1) FR_INST(N, 2) FR_ALIAS4(N)

#if KRIPKE_FR_GROUP == 0
FR_ALL(1) FR_ALL(2) FR_ALL(3) FR_ALL(4) FR_ALL(5) FR_ALL(6) FR_ALL(7)
#elif KRIPKE_FR_GROUP == 1
FR_ALL(8) FR_ALL(9) FR_ALL(10)
#elif KRIPKE_FR_GROUP == 2
FR_ALL(11) FR_ALL(12) FR_BIG(13)
#elif KRIPKE_FR_GROUP == 3
FR_BIG(14) FR_BIG(15) FR_BIG(16)
#endif

}  // namespace kripke
