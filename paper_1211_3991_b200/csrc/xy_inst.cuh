// xy_inst.cuh -- shared by the xy_inst_*.cu translation units: the switch from run-time (G, column blocks) to the
// k_phase / k_cycle template instantiation.
#pragma once
#include "xy_cycle.cuh"
#include "xy_dispatch.h"
#include "xy_sweep.cuh"

namespace xy {

// the k_phase<G, CB, MODE, W> instantiation for G lanes per site (CB = 0: R a multiple of 64 larger than 64)
template <int MODE, int W>
const void *phase_function_mode(int G, bool single_block) {
    switch (G) {
        case 32: return single_block ? reinterpret_cast<const void *>(k_phase<32, 1, MODE, W>)
                                     : reinterpret_cast<const void *>(k_phase<32, 0, MODE, W>);
        case 16: return reinterpret_cast<const void *>(k_phase<16, 1, MODE, W>);
        case 8: return reinterpret_cast<const void *>(k_phase<8, 1, MODE, W>);
        case 4: return reinterpret_cast<const void *>(k_phase<4, 1, MODE, W>);
        case 2: return reinterpret_cast<const void *>(k_phase<2, 1, MODE, W>);
        default: return reinterpret_cast<const void *>(k_phase<1, 1, MODE, W>);
    }
}

template <int ORDER>
const void *cycle_function_order(int G) {
    switch (G) {
        case 32: return reinterpret_cast<const void *>(k_cycle<32, ORDER>);
        case 16: return reinterpret_cast<const void *>(k_cycle<16, ORDER>);
        case 8: return reinterpret_cast<const void *>(k_cycle<8, ORDER>);
        case 4: return reinterpret_cast<const void *>(k_cycle<4, ORDER>);
        case 2: return reinterpret_cast<const void *>(k_cycle<2, ORDER>);
        default: return reinterpret_cast<const void *>(k_cycle<1, ORDER>);
    }
}

}  // namespace xy
