// xy_cycle.cuh -- k_cycle<G, ORDER, W>: whole PT cycles of ONE SAMPLE in ONE launch by ONE THREAD-BLOCK CLUSTER.
//
// The paper processes the colour classes "sequentially on each MCS" and pays for it with time ~ Q/2
// (PAPER.md:494); with one launch per colour class that is ~4 us of launch latency per class on B200, which bounds the
// small samples (BASELINE.json configs 0, 1 and the L <= 128 points of config 3's scan: a class is a few hundred rows).
// Samples never interact (Eq. 12), so the only ordering needed is BETWEEN THE COLOUR CLASSES OF ONE SAMPLE:
// a cluster of C CTAs (C <= 8) owns a sample, runs every colour class of every sweep of n_cycles cycles -- Metropolis,
// over-relaxation, the fused measurement, and the swap round -- and separates the classes with the HARDWARE cluster
// barrier (barrier.cluster.arrive.release / wait.acquire, ~0.2 us) instead of a kernel boundary.  No grid-wide barrier
// and no co-residency requirement: clusters are independent, a grid larger than the chip simply runs in waves.
//
// Everything a class does is the same code as the per-launch path (sweep_prep / sweep_phase / sweep_reduce_to_fx /
// sweep_finalize / pt_swap_sample, xy_sweep.cuh and xy_kernels.cuh) with the same Philox keying and the same exact
// integer reductions, so angles, labels, accumulators and counters are BIT-IDENTICAL to the k_phase path
// (tests/test_gpu_cycle.py).  Between arrive and wait a warp stages its share of the next class (graph data only),
// exactly what k_phase does between griddepcontrol.launch_dependents and griddepcontrol.wait.
//
// theta stays in global memory / L2 rather than in distributed shared memory: a DSMEM read costs as much as an L2 hit
// (~215 vs ~234-262 cycles) and DSMEM moves ~20 B/cycle/SM, less than what an SM draws from L2 here (B300_MICROARCH.md,
// "CGA; DSMEM"); the win of the cluster is the barrier, not the storage.  The acquire at cluster scope invalidates L1,
// so the cp.async.ca gathers of the next class see the neighbours' new angles.
//
// ORDER 0: sweep = Metropolis over all colours, then or_per_sweep x over-relaxation over all colours;
// ORDER 1: interleaved (Metropolis + over-relaxation of a class from one gather, xy_set_order).  R = 2G <= 64 only
// (one column block), or_per_sweep >= 1.
#pragma once
#include <type_traits>

#include "xy_sweep.cuh"

namespace xy {

struct CycleArgs {
    SweepArgs sa;          // part = the share table for C * W warps per sample (or nullptr: equal shares)
    SwapArgs sw;
    int n_cycles, sps, orps, me;
    int q_max;
    int do_swap;           // 1: xy_run (E for the swap round, swap at the end of every cycle); 0: xy_run_sweeps (bare sweeps)
};

__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

template <int G, int ORDER, int W>
__global__ void __launch_bounds__(W * 32, 1) k_cycle(const CycleArgs a) {
    extern __shared__ __align__(16) unsigned char s_raw[];
    SweepWarp *s_w = reinterpret_cast<SweepWarp *>(s_raw);
    const TileArgs &t = a.sa.t;

    SweepCtx x;
    x.s = t.s0 + blockIdx.y;
    x.lane = threadIdx.x & 31;
    x.warp = threadIdx.x >> 5;
    x.sub = x.lane / G;
    x.q = x.lane % G;
    x.lb = reinterpret_cast<float2 *>(t.theta) + static_cast<size_t>(x.s) * t.N * G + x.q;
    x.rec = t.rec + static_cast<size_t>(x.s) * t.N;
    x.sidx = s_w[x.warp].idx;
    x.ring_l = &s_w[x.warp].ring[0][0][x.lane];
    x.ring_s = static_cast<uint32_t>(__cvta_generic_to_shared(x.ring_l));
    const bool leader = blockIdx.x == 0;                 // cluster dims (C, 1, 1), grid (C, samples): rank = blockIdx.x

    x.fx = t.fx;

    const uint32_t sweep0 = t.counters[0], round0 = t.counters[1];
    int iacc[6] = {0, 0, 0, 0, 0, 0};
    // The sums of a finished sweep are converted by the leader while the other CTAs already run the next class, which
    // (interleaved order) may flush partial sums of the NEXT sweep: consecutive tallied sweeps alternate two buffers.
    long long *fx_done = nullptr;                        // sums waiting for the leader
    int finalize_pending = 0;                            // 1: convert the sums, 3: ... and add them to the accumulators

    auto finalize_if_pending = [&]() {
        if (finalize_pending) {
            if (leader) sweep_finalize(t, fx_done, x.s, (finalize_pending & 2) != 0);
            finalize_pending = 0;
        }
    };
    // one colour class: stage the share (graph data), wait until the cluster has finished the previous class, update.
    // The leader converts a finished sweep's sums right after the wait (all CTAs' atomics are visible then).
    auto phase = [&](auto mode, int colour, uint32_t sweep) {
        constexpr int MODE = decltype(mode)::value;
        const PhasePrep P = sweep_prep<G, 1>(a.sa, x, kModeOverrelax, colour, gridDim.x * W, blockIdx.x * W + x.warp, true);
        __syncwarp();
        cluster_wait();
        finalize_if_pending();
        sweep_phase<G, 1, MODE>(t, x, P, sweep, iacc);
        cluster_arrive();
    };
    // the sweep's E, Mx, My: per-lane partial sums -> the sample's 64-bit sums (the arrive of the class that follows
    // publishes them); the leader converts them after the next wait
    auto tally_done = [&](bool accumulate) {
        sweep_reduce_to_fx<G, W>(t, x, iacc, s_w);
#pragma unroll
        for (int c = 0; c < 6; ++c) iacc[c] = 0;
        __syncthreads();                                  // the ring slices served as scratch: done before the next staging
        finalize_pending = accumulate ? 3 : 1;
        fx_done = x.fx;
        x.fx = x.fx == t.fx ? t.fx + t.fx_stride : t.fx;   // the next tallied sweep adds to the other buffer
    };

    cluster_arrive();
    for (int cyc = 0; cyc < a.n_cycles; ++cyc) {
        for (int k = 1; k <= a.sps; ++k) {
            const uint32_t sweep = sweep0 + static_cast<uint32_t>(cyc * a.sps + k);
            const bool measured = a.do_swap && a.me > 0 && sweep % static_cast<uint32_t>(a.me) == 0u;
            const bool need_e = a.do_swap && (measured || k == a.sps);
            if constexpr (ORDER == 0) {
                for (int c = 0; c < a.q_max; ++c) phase(std::integral_constant<int, kModeMetropolis>{}, c, sweep);
                for (int o = 0; o < a.orps; ++o) {
                    if (need_e && o == a.orps - 1) {
                        // tally in the arrive-to-wait window of the LAST class: split the phase by hand
                        for (int c = 0; c < a.q_max; ++c) {
                            const PhasePrep P = sweep_prep<G, 1>(a.sa, x, kModeOverrelax, c, gridDim.x * W, blockIdx.x * W + x.warp, true);
                            __syncwarp();
                            cluster_wait();
                            finalize_if_pending();
                            sweep_phase<G, 1, kModeOrMeasure>(t, x, P, sweep, iacc);
                            if (c == a.q_max - 1) tally_done(measured);
                            cluster_arrive();
                        }
                    } else {
                        for (int c = 0; c < a.q_max; ++c) phase(std::integral_constant<int, kModeOverrelax>{}, c, sweep);
                    }
                }
            } else {
                for (int c = 0; c < a.q_max; ++c) {
                    if (need_e) {
                        const PhasePrep P = sweep_prep<G, 1>(a.sa, x, kModeOverrelax, c, gridDim.x * W, blockIdx.x * W + x.warp, true);
                        __syncwarp();
                        cluster_wait();
                        finalize_if_pending();
                        sweep_phase<G, 1, kModeMetOrMeasure>(t, x, P, sweep, iacc);
                        if (c == a.q_max - 1) tally_done(measured);
                        cluster_arrive();
                    } else {
                        phase(std::integral_constant<int, kModeMetOr>{}, c, sweep);
                    }
                }
            }
        }
        if (a.do_swap) {
            // end of the cycle: the leader converts the last sweep's sums and makes the swap round; the arrive that
            // follows publishes the new beta / width per slot to the whole cluster before the next Metropolis class
            cluster_wait();
            if (leader) {
                sweep_finalize(t, fx_done, x.s, (finalize_pending & 2) != 0);
                __syncthreads();
                pt_swap_sample(a.sw, x.s, round0 + static_cast<uint32_t>(cyc));
            }
            finalize_pending = 0;
            cluster_arrive();
        }
    }
    cluster_wait();
}

}  // namespace xy
