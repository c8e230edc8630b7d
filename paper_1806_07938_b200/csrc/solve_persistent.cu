// solve_persistent.cu -- persistent cooperative solver (one kernel per solve, device-side grid barriers).
#include "tomo.h"
#include "tomo_plan.hpp"

namespace tomo {
int solve_persistent(tomo_plan *, const float *, float *, int, int, const float *, cudaStream_t) {
    set_error("persistent solver not built yet");
    return TOMO_EUNSUPPORTED;
}
}  // namespace tomo
