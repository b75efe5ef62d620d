// xy_diag.cuh -- L2 bandwidth microbenchmarks behind xy_l2_bandwidth (include/xy_b200.h): the roofline denominator for
// the sample groups that the time-blocked schedule keeps resident in the 126 MB L2 (BASELINE.json north_star: "achieved
// HBM GB/s, or L2 GB/s when the state fits in the 126 MB L2 ... against the chip's peak"; "L2 peak is
// not in MEASURED_PEAKS.json -- measure it with a streaming-read microbenchmark on a 32 MB buffer").
//
// k_l2_stream: every CTA reads its own contiguous slice of the buffer `passes` times with 16-byte ld.global.cg loads
//   (L1 bypassed, so every pass is served by L2), eight independent loads in flight per thread.
// k_l2_gather: the access shape of the neighbour gather of k_phase at R = 64 -- a warp reads one aligned 256-byte row
//   (8 bytes per lane) at a pseudo-random row index, eight rows in flight per warp -- so the number says what L2 gives
//   for random 256-byte requests rather than for a linear stream.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace xy {

__global__ void __launch_bounds__(512) k_l2_stream(const uint4 *buf, size_t n_vec /*uint4 per CTA slice*/, int passes,
                                                   unsigned *sink) {
    const uint4 *p = buf + static_cast<size_t>(blockIdx.x) * n_vec;
    unsigned acc = 0u;
    for (int pass = 0; pass < passes; ++pass) {
        for (size_t i = threadIdx.x; i < n_vec; i += 8 * blockDim.x) {
            uint4 v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const size_t k = i + static_cast<size_t>(u) * blockDim.x;
                v[u] = k < n_vec ? __ldcg(p + k) : make_uint4(0u, 0u, 0u, 0u);
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) acc ^= v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
        }
    }
    if (acc == 0x9e3779b9u) sink[0] = acc;      // never true for the zero-filled buffer: keeps the loads alive
}

__global__ void __launch_bounds__(512) k_l2_gather(const uint2 *buf, uint32_t n_rows /*256-byte rows, a power of two*/,
                                                   int rows_per_warp, unsigned *sink) {
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    uint32_t state = gw * 2654435761u + 12345u;
    unsigned acc = 0u;
    for (int i = 0; i < rows_per_warp; i += 8) {
        uint2 v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            state = state * 1664525u + 1013904223u;                       // warp-uniform LCG: one row per request
            const uint32_t row = (state >> 8) & (n_rows - 1u);
            v[u] = __ldcg(buf + static_cast<size_t>(row) * 32u + lane);
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) acc ^= v[u].x ^ v[u].y;
    }
    if (acc == 0x9e3779b9u) sink[0] = acc;
}

}  // namespace xy
