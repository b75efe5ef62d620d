// k_phase<G, CB, MODE, W = 8> for MODE in {3, 4, 5} (see xy_dispatch.h)
#include "xy_inst.cuh"

namespace xy {
const void *phase_function_w8_b(int G, bool single_block, int mode) {
    return mode == 3 ? phase_function_mode<3, 8>(G, single_block)
         : mode == 4 ? phase_function_mode<4, 8>(G, single_block)
         : mode == 5 ? phase_function_mode<5, 8>(G, single_block) : nullptr;
}
}  // namespace xy
