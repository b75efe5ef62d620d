// xy_dispatch.h -- host-side lookup of the k_phase / k_cycle instantiations.  The kernels are templates (xy_sweep.cuh,
// xy_cycle.cuh); their instantiations are spread over several translation units (xy_inst_*.cu) so that the library
// builds in parallel; xy_b200.cu only sees these function-pointer lookups.
#pragma once

namespace xy {

constexpr int kCycleWarps = 8;       // warps per CTA of k_cycle: 256 threads x 128 registers (no spills, all gathers of a row in
                                     // flight), two CTAs per SM.  Measured: 16 warps x 64 registers (134 B of spills, twice the warps
                                     // per sample) gives the same throughput
constexpr int kCycleMaxCtas = 16;    // largest cluster of k_cycle (the non-portable size)
constexpr int kCycleMaxQ = 12;       // most colours a sample may have on the cluster path
constexpr int kCycleAutoRows = 36;   // automatic path choice: cluster path while a warp owns at most this many rows

// k_phase<G, CB, MODE, W> for W in {8, 32} (MODE 0..5), W = 28 (MODE 3) and W = 24 (MODE 5); CB = single_block ? 1 : 0 (G = 32 only).
// nullptr for a combination that is not built.
const void *phase_function(int W, int G, bool single_block, int mode);
// k_cycle<G, ORDER>
const void *cycle_function(int order, int G);

// per translation unit
const void *phase_function_w8_a(int G, bool single_block, int mode);    // modes 0, 1, 2
const void *phase_function_w8_b(int G, bool single_block, int mode);    // modes 3, 4, 5
const void *phase_function_w32_a(int G, bool single_block, int mode);
const void *phase_function_w32_b(int G, bool single_block, int mode);
const void *phase_function_w24(int G, bool single_block, int mode);     // modes 3, 5
const void *cycle_function_o0(int G);
const void *cycle_function_o1(int G);

}  // namespace xy
