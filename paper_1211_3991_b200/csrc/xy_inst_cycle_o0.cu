// k_cycle<G, ORDER = 0> (see xy_dispatch.h)
#include "xy_inst.cuh"

namespace xy {
const void *cycle_function_o0(int G) { return cycle_function_order<0>(G); }
}  // namespace xy
