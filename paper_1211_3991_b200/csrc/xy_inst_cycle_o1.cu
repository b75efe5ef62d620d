// k_cycle<G, ORDER = 1> (see xy_dispatch.h)
#include "xy_inst.cuh"

namespace xy {
const void *cycle_function_o1(int G) { return cycle_function_order<1>(G); }
}  // namespace xy
