// k_phase<G, CB, MODE, W = 24> for the measuring modes 3 and 5 (see xy_dispatch.h)
#include "xy_inst.cuh"

namespace xy {
const void *phase_function_w24(int G, bool single_block, int mode) {
    return mode == 3 ? phase_function_mode<3, 24>(G, single_block) : mode == 5 ? phase_function_mode<5, 24>(G, single_block) : nullptr;
}
}  // namespace xy
