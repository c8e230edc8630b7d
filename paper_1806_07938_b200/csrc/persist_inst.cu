// persist_inst.cu -- one translation unit per FFT edge: compiled with -DTOMO_PINST=<P>, instantiates the persistent
// kernel for the three precisions (include/tomo.h: TOMO_F32, TOMO_F32S_F64A, TOMO_F64) at that size.
#include "persist_host.cuh"

#ifndef TOMO_PINST
#error "compile with -DTOMO_PINST=<FFT edge>"
#endif

namespace tomo {

template <> int persist_run<TOMO_PINST>(tomo_plan *pl, cudaStream_t st, const PLaunch &L) {
    if (pl->opt.precision == TOMO_F32) return persist_launch<float, float, TOMO_PINST>(pl, st, L);
    if (pl->opt.precision == TOMO_F32S_F64A) return persist_launch<double, float, TOMO_PINST>(pl, st, L);
    return persist_launch<double, double, TOMO_PINST>(pl, st, L);
}

}  // namespace tomo
