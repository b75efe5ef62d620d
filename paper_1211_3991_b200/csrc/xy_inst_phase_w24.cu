// k_phase<G, CB, MODE, W> for the measuring modes: MODE 3 with W = 28 warps (72 registers, no spills), MODE 5 with W = 24
// (80 registers; at 72 it spills ~100 bytes) -- see xy_dispatch.h
#include "xy_inst.cuh"

namespace xy {
const void *phase_function_w24(int G, bool single_block, int mode) {
    return mode == 3 ? phase_function_mode<3, 28>(G, single_block) : mode == 5 ? phase_function_mode<5, 24>(G, single_block) : nullptr;
}
}  // namespace xy
