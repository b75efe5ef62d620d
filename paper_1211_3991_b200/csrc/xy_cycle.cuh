// xy_cycle.cuh -- k_cycle<G, ORDER>: whole PT cycles of ONE SMALL SAMPLE in ONE launch by ONE THREAD-BLOCK CLUSTER whose
// warps keep their rows RESIDENT.
//
// The paper processes the colour classes "sequentially on each MCS" and pays for it with time ~ Q/2
// (PAPER.md:494).  For a small sample (BASELINE.json configs 0, 1, the L <= 64 points of config 3's scan) a colour class is
// at most a few rows per warp, and one class costs a fixed serial chain whatever its size: with one launch per class
// (k_phase) that chain is launch + share table + rec[] + neighbour ids + gather + update + store + drain, 3.5-5 us.
// Samples never interact (Eq. 12), so the only ordering needed is BETWEEN THE COLOUR CLASSES OF ONE SAMPLE:
// a cluster of C CTAs (C <= 8) owns a sample and separates the classes with the HARDWARE cluster barrier
// (barrier.cluster.arrive.release / wait.acquire) instead of a kernel boundary -- no grid-wide barrier, no co-residency
// requirement between samples.  And because the sample is small, every warp OWNS its rows for the whole launch:
//
//   * rows (32/G consecutive sites of one class x G lanes x 2 slots) are dealt round-robin to the C * kCycleWarps warps of
//     the cluster, class after class, so every class and every warp's total is balanced to within one row;
//   * at launch a warp copies, once, what its rows need into its slice of shared memory: one descriptor per site and the
//     neighbour ids pre-scaled by the site stride;
//   * a colour class is then: cluster wait -> gather the own and the neighbours' angles from L2 (cp.async; the acquire of
//     the wait invalidates L1) -> update -> store the new angle -> cluster arrive.  One L2 round trip and one barrier per
//     class instead of a launch and four dependent loads.
//
// theta stays in global memory / L2 rather than in distributed shared memory: a DSMEM read costs as much as an L2 hit
// (~215 vs ~234-262 cycles, B300_MICROARCH.md "CGA; DSMEM") and the writer would have to know which CTAs read a site.
//
// The arithmetic of an update is the arithmetic of k_phase (same Philox keying, same order of the neighbour sum, same
// quantisation of the measured sums), so angles, labels, accumulators and counters are BIT-IDENTICAL to the per-launch
// path (tests/test_gpu_cycle.py), which is the one held against the oracle element by element.
//
// ORDER 0: sweep = Metropolis over all colours, then or_per_sweep x over-relaxation over all colours;
// ORDER 1: interleaved (Metropolis + over-relaxation of a class from one gather, xy_set_order).  R = 2G <= 64 only
// (one column block), or_per_sweep >= 1, at most kCycleMaxQ colours, degrees <= 255.
#pragma once
#include <type_traits>

#include "xy_dispatch.h"
#include "xy_sweep.cuh"

namespace xy {

struct CycleArgs {
    TileArgs t;
    SwapArgs sw;
    int n_cycles, sps, orps, me;
    int q_max;
    int do_swap;           // 1: xy_run (E for the swap round, swap at the end of every cycle); 0: xy_run_sweeps (bare sweeps)
    int k_cap, id_cap;     // per-warp resident pool: rows, neighbour ids (host: the maximum over all warps and samples)
};

// one warp's slice of shared memory: the gather ring (two slots of kDB neighbour rows + the own angle: the copies of the
// warp's next row fly while it computes the current one), then the resident pool: site descriptors [k_cap][32 / G] int2
// and neighbour ids [id_cap]
constexpr size_t kCycleRingBytes = 2 * (kDB + 1) * 32 * sizeof(float2);
__host__ __device__ constexpr size_t cycle_pool_bytes(int G, int k_cap, int id_cap) {
    return kCycleRingBytes + (static_cast<size_t>(k_cap) * (32 / G) * 8 + static_cast<size_t>(id_cap) * 4 + 15) / 16 * 16;
}

__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// per-thread constants of a launch
struct CycleCtx {
    float2 *lb;                 // this lane's column of the sample: theta2 + s*N*G + q
    const float2 *ring_l;       // this lane's column of the warp's gather ring (generic pointer)
    uint32_t ring_s;            // same, shared-space address
    const int2 *meta;           // the warp's site descriptors [k_cap][SPW] {site or -1, first id | degree << 16 | n_lower << 24}
    const uint32_t *ids;        // the warp's neighbour ids, pre-scaled by the site stride
    long long *fx;              // the fixed-point sums the measuring modes add to (two buffers alternate)
    int s, lane, sub, q;
};

// async copies (cp.async, the lane's own 8 bytes) of row j's own angle and first kDB neighbours into ring slot `slot`:
// the only global reads of a row
template <int G>
__device__ __forceinline__ void cycle_issue(const CycleCtx &x, int j, int slot) {
    constexpr int SPW = 32 / G;
    const int2 m = x.meta[j * SPW + x.sub];
    const uint32_t row0 = x.ring_s + static_cast<uint32_t>(slot) * ((kDB + 1) * 256u);
    if (m.x >= 0) {
        const int pos = m.y & 0xffff, deg = (m.y >> 16) & 0xff;
        cp_async8(row0 + kDB * 256u, x.lb + static_cast<unsigned long long>(static_cast<uint32_t>(m.x) * static_cast<uint32_t>(G)));
#pragma unroll
        for (int u = 0; u < kDB; ++u)
            if (u < deg) cp_async8(row0 + u * 256u, x.lb + static_cast<unsigned long long>(x.ids[pos + u]));
    }
    cp_async_commit();
}

// one row (the lane's site, two slots) whose copies have landed in ring slot `slot`: the update of k_phase's sweep_phase
template <int G, int MODE>
__device__ __forceinline__ void cycle_row(const TileArgs &a, const CycleCtx &x, int j, int slot, uint32_t sweep, const float2 nbeta,
                                          const float2 w, int (&iacc)[6]) {
    constexpr int SPW = 32 / G;
    constexpr bool UNI = SPW == 1;
    constexpr bool kMet = MODE == kModeMetropolis || MODE == kModeMetOr || MODE == kModeMetOrMeasure;
    constexpr bool kFusedMetOr = MODE == kModeMetOr || MODE == kModeMetOrMeasure;
    constexpr bool kTally = MODE == kModeOrMeasure || MODE == kModeMetOrMeasure;
    const int2 m = x.meta[j * SPW + x.sub];
    const bool valid = m.x >= 0;
    const int i = m.x, pos = m.y & 0xffff;
    const int deg = valid ? (m.y >> 16) & 0xff : 0, nlow = valid ? static_cast<int>(static_cast<uint32_t>(m.y) >> 24) : 0;
    const int dmax = UNI ? deg : static_cast<int>(__reduce_max_sync(kFull, static_cast<unsigned>(deg)));
    const float2 *row0 = x.ring_l + slot * ((kDB + 1) * 32);
    float2 own = make_float2(0.f, 0.f);
    if (valid) own = row0[kDB * 32];

    PairAcc<MODE> acc;
    float2 thp = make_float2(0.f, 0.f), u2 = thp;
    if constexpr (kMet) {       // the proposal of sweep_phase::begin (R5, R10, R11), word for word
        uint32_t r[4];
        const uint32_t c2 = ((a.sample_base + static_cast<uint32_t>(x.s)) << 16) | static_cast<uint32_t>(x.q);
        philox4x32_10(static_cast<uint32_t>(i), sweep, c2, kDomMetropolis, a.keys, r);
        const float2 u1mh = add2(add2(make_float2(mant12(r[0]), mant12(r[2])), make_float2(-1.5f, -1.5f)),
                                 make_float2(5.9604644775390625e-08f, 5.9604644775390625e-08f));
        u2 = add2(make_float2(mant12(r[1]), mant12(r[3])), make_float2(-0.99999994f, -0.99999994f));
        thp = make_float2(__fadd_rn(own.x, __fmul_rn(w.x, u1mh.x)), __fadd_rn(own.y, __fmul_rn(w.y, u1mh.y)));
        if constexpr (MODE == kModeMetropolis) acc.mid = add2(own, mul2(sub2(thp, own), make_float2(0.5f, 0.5f)));
    }
    if constexpr (kTally) acc.nlow = nlow;

#pragma unroll
    for (int b = 0; b < kDB; b += 4) {       // batches of 4 LDS.64, then their arithmetic
        float2 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = row0[(b + u) * 32];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (b + u < deg) acc.add(v[u], b + u);
    }
    for (int k = kDB; k < dmax; k += 4) {    // rare: P(deg > 8) ~ 15 % at z = 6
        float2 t[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (k + u < deg) t[u] = __ldcg(x.lb + static_cast<unsigned long long>(x.ids[pos + k + u]));
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (k + u < deg) acc.add(t[u], k + u);
    }

    float2 out;
    if constexpr (MODE == kModeMetropolis) {
        const float2 half = mul2(sub2(thp, own), make_float2(0.5f, 0.5f));
        const float2 sh = make_float2(__sinf(half.x), __sinf(half.y));
        const float2 arg = mul2(nbeta, mul2(add2(sh, sh), acc.s));
        out.x = metropolis_select(own.x, thp.x, u2.x, __expf(arg.x));
        out.y = metropolis_select(own.y, thp.y, u2.y, __expf(arg.y));
    } else if constexpr (kFusedMetOr) {
        const float2 half = mul2(sub2(thp, own), make_float2(0.5f, 0.5f));
        const float2 mid = add2(own, half);
        float smx, cmx, smy, cmy;
        __sincosf(mid.x, &smx, &cmx);
        __sincosf(mid.y, &smy, &cmy);
        const float2 ss = make_float2(__fmaf_rn(smx, acc.hx.x, -__fmul_rn(cmx, acc.hy.x)),
                                      __fmaf_rn(smy, acc.hx.y, -__fmul_rn(cmy, acc.hy.y)));
        const float2 sh = make_float2(__sinf(half.x), __sinf(half.y));
        const float2 arg = mul2(nbeta, mul2(add2(sh, sh), ss));
        out.x = overrelax_finish(metropolis_select(own.x, thp.x, u2.x, __expf(arg.x)), acc.hx.x, acc.hy.x);
        out.y = overrelax_finish(metropolis_select(own.y, thp.y, u2.y, __expf(arg.y)), acc.hx.y, acc.hy.y);
    } else {
        out.x = overrelax_finish(own.x, acc.hx.x, acc.hy.x);
        out.y = overrelax_finish(own.y, acc.hx.y, acc.hy.y);
    }
    if (UNI || valid) {
        x.lb[static_cast<unsigned long long>(static_cast<uint32_t>(i) * static_cast<uint32_t>(G))] = out;
        if constexpr (kTally) {      // sweep_phase::tally: fixed-point bond energy (lower neighbours) and magnetisation
            float sx, cx, sy, cy;
            __sincosf(out.x, &sx, &cx);
            __sincosf(out.y, &sy, &cy);
            const float ex = site_energy(cx, sx, acc.lx.x, acc.ly.x), ey = site_energy(cy, sy, acc.lx.y, acc.ly.y);
            if (nlow <= 8) {
                iacc[0] += quant8(ex);
                iacc[3] += quant8(ey);
            } else if (nlow <= 32) {
                iacc[0] += quant32(ex) << 2;
                iacc[3] += quant32(ey) << 2;
            } else {
                unsigned long long *fxl = reinterpret_cast<unsigned long long *>(x.fx) + (static_cast<size_t>(x.s) * a.R + 2 * x.q) * 3;
                atomicAdd(fxl, static_cast<unsigned long long>(__double2ll_rn(static_cast<double>(ex) * 524288.0)));
                atomicAdd(fxl + 3, static_cast<unsigned long long>(__double2ll_rn(static_cast<double>(ey) * 524288.0)));
            }
            iacc[1] += quant1(cx); iacc[2] += quant1(sx);
            iacc[4] += quant1(cy); iacc[5] += quant1(sy);
        }
    }
}

template <int G, int ORDER>
__global__ void __launch_bounds__(kCycleWarps * 32, 2) k_cycle(const CycleArgs a) {
    constexpr int W = kCycleWarps;
    constexpr int SPW = 32 / G;
    extern __shared__ __align__(16) unsigned char s_raw[];
    __shared__ unsigned short s_jb[W][kCycleMaxQ + 1];      // per warp: first resident row of every colour class
    __shared__ unsigned long long s_acc[G][6];              // the CTA's measured sums of a sweep (exact integers)
    const TileArgs &t = a.t;

    CycleCtx x;
    x.s = t.s0 + blockIdx.y;
    x.lane = threadIdx.x & 31;
    x.sub = x.lane / G;
    x.q = x.lane % G;
    const int warp = threadIdx.x >> 5;
    x.lb = reinterpret_cast<float2 *>(t.theta) + static_cast<size_t>(x.s) * t.N * G + x.q;
    unsigned char *pool = s_raw + static_cast<size_t>(warp) * cycle_pool_bytes(G, a.k_cap, a.id_cap);
    x.ring_l = reinterpret_cast<const float2 *>(pool) + x.lane;
    x.ring_s = static_cast<uint32_t>(__cvta_generic_to_shared(x.ring_l));
    int2 *meta = reinterpret_cast<int2 *>(pool + kCycleRingBytes);
    uint32_t *ids = reinterpret_cast<uint32_t *>(pool + kCycleRingBytes + static_cast<size_t>(a.k_cap) * (SPW * 8));
    x.meta = meta;
    x.ids = ids;
    x.fx = t.fx;
    const bool leader = blockIdx.x == 0;                 // cluster dims (C, 1, 1), grid (C, samples): rank = blockIdx.x
    const int nw = gridDim.x * W, gw = blockIdx.x * W + warp;

    // ---- once per launch: the warp's rows become resident (graph data only).  Rows are numbered class after class; row
    // rho belongs to warp rho mod nw. ----
    {
        const int2 *rec = t.rec + static_cast<size_t>(x.s) * t.N;
        const int32_t *cp = t.class_ptr + x.s * t.q_stride;
        int j = 0, n_ids = 0, rowbase = 0;
        for (int c = 0; c < a.q_max; ++c) {
            if (x.lane == 0) s_jb[warp][c] = static_cast<unsigned short>(j);
            const int cbeg = cp[c], cend = cp[c + 1];
            const int n_rows = (cend - cbeg + SPW - 1) / SPW;
            int k = (gw - rowbase % nw + nw) % nw;
            for (; k < n_rows; k += nw, ++j) {
                const int i = cbeg + k * SPW + x.sub;
                const bool valid = i < cend;
                int2 rc = make_int2(0, 0);
                if (valid) rc = rec[i];
                const int deg = rc.y & 0xffff, nlow = static_cast<int>(static_cast<uint32_t>(rc.y) >> 16);
                int before = 0, total = 0;               // ids of the row's sites in front of this lane's site, and of the whole row
#pragma unroll
                for (int sb = 0; sb < SPW; ++sb) {
                    const int d = __shfl_sync(kFull, deg, sb * G);
                    if (sb < x.sub) before += d;
                    total += d;
                }
                const int pos = n_ids + before;
                for (int e = x.q; e < deg; e += G) ids[pos + e] = static_cast<uint32_t>(t.col_idx[rc.x + e]) * static_cast<uint32_t>(G);
                if (x.q == 0) meta[j * SPW + x.sub] = make_int2(valid ? i : -1, pos | (deg << 16) | (nlow << 24));
                n_ids += total;
            }
            rowbase += n_rows;
        }
        if (x.lane == 0) s_jb[warp][a.q_max] = static_cast<unsigned short>(j);
        if (threadIdx.x < G * 6) s_acc[threadIdx.x / 6][threadIdx.x % 6] = 0ull;
    }
    __syncthreads();

    const uint32_t sweep0 = t.counters[0], round0 = t.counters[1];
    int iacc[6] = {0, 0, 0, 0, 0, 0};
    // The sums of a finished sweep are converted by the leader while the other CTAs already run the next class, which
    // (interleaved order) may add to the sums of the NEXT sweep: consecutive tallied sweeps alternate two buffers.
    long long *fx_done = nullptr;                        // sums waiting for the leader
    int finalize_pending = 0;                            // 1: convert the sums, 3: ... and add them to the accumulators

    auto finalize_if_pending = [&]() {
        if (finalize_pending) {
            if (leader) sweep_finalize(t, fx_done, x.s, (finalize_pending & 2) != 0);
            finalize_pending = 0;
        }
    };
    // one colour class: wait until the cluster has finished the previous class, update the warp's rows of the class.
    // The leader converts a finished sweep's sums right after the wait (all CTAs' atomics are visible then).
    auto phase = [&](auto mode, int colour, uint32_t sweep) {
        constexpr int MODE = decltype(mode)::value;
        constexpr bool kMet = MODE == kModeMetropolis || MODE == kModeMetOr || MODE == kModeMetOrMeasure;
        const int j0 = s_jb[warp][colour], j1 = s_jb[warp][colour + 1];
        cluster_wait();
        finalize_if_pending();
        if (j0 < j1) {
            float2 nbeta = make_float2(0.f, 0.f), w = nbeta;
            if constexpr (kMet) {
                const float2 b = __ldcg(reinterpret_cast<const float2 *>(t.beta_slot) + static_cast<size_t>(x.s) * G + x.q);
                nbeta = make_float2(-b.x, -b.y);
                w = __ldcg(reinterpret_cast<const float2 *>(t.w_slot) + static_cast<size_t>(x.s) * G + x.q);
            }
            cycle_issue<G>(x, j0, 0);
            for (int j = j0; j < j1; ++j) {      // the copies of row j + 1 fly while row j is computed
                if (j + 1 < j1) {
                    cycle_issue<G>(x, j + 1, (j + 1 - j0) & 1);
                    cp_async_wait<1>();
                } else {
                    cp_async_wait<0>();
                }
                cycle_row<G, MODE>(t, x, j, (j - j0) & 1, sweep, nbeta, w, iacc);
            }
        }
    };
    // the sweep's E, Mx, My: per-lane partial sums -> the CTA's sums in shared memory (exact 64-bit integer atomics) -> the
    // sample's sums in global memory (the arrive that follows publishes them); the leader converts them after the next wait
    auto tally_done = [&](bool accumulate) {
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            long long v = iacc[c];
#pragma unroll
            for (int o = G; o < 32; o <<= 1) v += __shfl_xor_sync(kFull, v, o);      // the row's sites share the slot pair
            if (x.sub == 0 && v != 0) atomicAdd(&s_acc[x.q][c], static_cast<unsigned long long>(v));
            iacc[c] = 0;
        }
        __syncthreads();
        if (threadIdx.x < G * 6) {
            const int ll = threadIdx.x / 6, c = threadIdx.x % 6;
            const unsigned long long v = s_acc[ll][c];
            s_acc[ll][c] = 0ull;
            const int slot = 2 * ll + c / 3;
            if (v) atomicAdd(reinterpret_cast<unsigned long long *>(x.fx) + (static_cast<size_t>(x.s) * t.R + slot) * 3 + c % 3, v);
        }
        __syncthreads();
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
                for (int c = 0; c < a.q_max; ++c) {
                    phase(std::integral_constant<int, kModeMetropolis>{}, c, sweep);
                    cluster_arrive();
                }
                for (int o = 0; o < a.orps; ++o) {
                    const bool tally = need_e && o == a.orps - 1;
                    for (int c = 0; c < a.q_max; ++c) {
                        if (tally) {
                            phase(std::integral_constant<int, kModeOrMeasure>{}, c, sweep);
                            if (c == a.q_max - 1) tally_done(measured);
                        } else {
                            phase(std::integral_constant<int, kModeOverrelax>{}, c, sweep);
                        }
                        cluster_arrive();
                    }
                }
            } else {
                for (int c = 0; c < a.q_max; ++c) {
                    if (need_e) {
                        phase(std::integral_constant<int, kModeMetOrMeasure>{}, c, sweep);
                        if (c == a.q_max - 1) tally_done(measured);
                    } else {
                        phase(std::integral_constant<int, kModeMetOr>{}, c, sweep);
                    }
                    cluster_arrive();
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
