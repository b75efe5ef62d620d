// k_phase<G, CB, MODE, W = 32> for MODE in {0, 1, 2} (see xy_dispatch.h)
#include "xy_inst.cuh"

namespace xy {
const void *phase_function_w32_a(int G, bool single_block, int mode) {
    return mode == 0 ? phase_function_mode<0, 32>(G, single_block)
         : mode == 1 ? phase_function_mode<1, 32>(G, single_block)
         : mode == 2 ? phase_function_mode<2, 32>(G, single_block) : nullptr;
}
}  // namespace xy
