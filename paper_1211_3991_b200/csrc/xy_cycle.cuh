// xy_cycle.cuh -- k_cycle<G, ORDER>: whole PT cycles of ONE SMALL SAMPLE in ONE launch by ONE THREAD-BLOCK CLUSTER that
// keeps the sample's angles in its DISTRIBUTED SHARED MEMORY.
//
// The paper processes the colour classes "sequentially on each MCS" and pays for it with time ~ Q/2
// (PAPER.md:494).  For a small sample (BASELINE.json configs 0, 1, the L <= 64 points of config 3's scan) a colour class is
// at most a few rows per warp, and one class costs a fixed serial chain whatever its size.  Measured on B200 (clock64
// stamps): with one launch per class (k_phase) the chain is launch + share table + rec[] + neighbour ids +
// gather + update + drain, 3.5-5 us; with a cluster barrier instead of the launch but the angles still in L2 it is
// barrier.cluster.arrive.release (~1100 cycles: the release drains the stores to L2) + wait + gather (~1300 cycles: one
// L2 round trip through cp.async) + update, ~3 us.  Both are memory round trips, not arithmetic.
// Samples never interact (Eq. 12), so the only ordering needed is BETWEEN THE COLOUR CLASSES OF ONE SAMPLE,
// and a small sample fits the shared memory of a few SMs.  So a cluster of C CTAs (C <= 8) owns a sample for the whole
// launch:
//
//   * every CTA owns a contiguous C-th of the rows (32/G consecutive sites x G lanes x 2 slots) of EVERY colour class --
//     the same region of the lattice in every class, so most neighbours are in the CTA's own shared memory -- and deals
//     them round-robin to its warps, class after class: every class and every warp's total is balanced to within a row;
//   * at launch a warp copies, once, what its rows need into its slice of shared memory: the rows' angles, one descriptor
//     per site, and for every neighbour WHERE ITS ANGLE LIVES: the rank of the owner's CTA and the offset in its shared
//     memory (closed forms, no table);
//   * a colour class is then: cluster wait -> gather the neighbours' angles from the owners' shared memory
//     (mapa + ld.shared::cluster: ~200 cycles instead of an L2 round trip) -> update -> write the new angle to the warp's
//     OWN shared memory -> cluster arrive.  No global memory access at all between two swap rounds: the measured sums of
//     a sweep are reduced in shared memory (exact integers), collected by the leader CTA through DSMEM and filed in its
//     resident copy of the accumulators; the angles and accumulators go back to global memory when the launch ends.
//
// The arithmetic of an update is the arithmetic of k_phase (same Philox keying, same order of the neighbour sum, same
// quantisation of the measured sums, same conversion), so angles, labels, accumulators and counters are BIT-IDENTICAL to
// the per-launch path (tests/test_gpu_cycle.py), which is the one held against the oracle element by element.
//
// ORDER 0: sweep = Metropolis over all colours, then or_per_sweep x over-relaxation over all colours;
// ORDER 1: interleaved (Metropolis + over-relaxation of a class from one gather, xy_set_order).  R = 2G <= 64 only
// (one column block), or_per_sweep >= 1, at most kCycleMaxQ colours, degrees <= 255, and the sample must fit the
// cluster's shared memory (the host plans this: cycle_plan in xy_b200.cu).
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

// one warp's slice of shared memory: its rows' angles [k_cap][32] float2, site descriptors [k_cap][32 / G] int2 and
// neighbour descriptors [id_cap] uint32 (the shared::cluster address of the neighbour's angles, slot pair 0)
__host__ __device__ constexpr size_t cycle_pool_bytes(int G, int k_cap, int id_cap) {
    return (static_cast<size_t>(k_cap) * (256 + (32 / G) * 8) + static_cast<size_t>(id_cap) * 4 + 15) / 16 * 16;
}

// first row of a class of n_rows rows that CTA b of n_cta owns: ceil(b n_rows / n_cta) (host and device)
__host__ __device__ constexpr int cycle_first_row(int b, int n_rows, int n_cta) {
    return static_cast<int>((static_cast<long long>(b) * n_rows + n_cta - 1) / n_cta);
}

__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
// The arrive between two colour classes publishes SHARED-MEMORY writes only (the warp's new angles and the CTA's measured
// sums live in its own shared memory, which the other CTAs of the cluster read directly, without a cache in between).
// barrier.cluster.arrive.release compiles to MEMBAR.ALL.GPU + ERRBAR (measured: ~1150 cycles per class, as much as the
// update itself); a CTA-scope fence (MEMBAR.ALL.CTA: the thread's shared-memory writes are performed) followed by the
// relaxed arrive orders the same shared-memory traffic for ~100 cycles.  Global-memory traffic between CTAs (the new beta
// per slot after a swap round) goes through the full release / acquire pair above.
__device__ __forceinline__ void cluster_arrive_shared() {
    __threadfence_block();
    asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");
}

// distributed shared memory: the same shared-memory address in the CTA of rank `rank`
__device__ __forceinline__ uint32_t cluster_map(uint32_t local_addr, uint32_t rank) {
    uint32_t ra;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(local_addr), "r"(rank));
    return ra;
}
// a neighbour's angles by shared::cluster address (mapped once, at launch; an address of the CTA's own shared-memory
// window is a valid shared::cluster address of this CTA)
__device__ __forceinline__ float2 ldc_f2(uint32_t cluster_addr) {
    float2 v;
    asm volatile("ld.shared::cluster.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(cluster_addr) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_cluster_u64(uint32_t local_addr, uint32_t rank) {
    unsigned long long v;
    asm volatile("ld.shared::cluster.u64 %0, [%1];" : "=l"(v) : "r"(cluster_map(local_addr, rank)) : "memory");
    return v;
}

// per-thread constants of a launch
struct CycleCtx {
    float2 *lb;                 // this lane's column of the sample in global memory: theta2 + s*N*G + q (load and write-back)
    float2 *own;                // this lane's column of the warp's resident rows: [k_cap], stride 32
    const int2 *meta;           // the warp's site descriptors [k_cap][SPW] {site or -1, first id | degree << 16 | n_lower << 24}
    const uint32_t *ids;        // the warp's neighbour descriptors: shared::cluster address of the neighbour's angles, slot pair 0
    uint32_t q8;                // 8 q: the lane's slot pair inside a site's 8 G bytes
    unsigned long long *sacc;   // the CTA's measured sums of the sweep being tallied [G][6]
    int s, lane, sub, q;
};

// one row (the lane's site, two slots): the update of k_phase's sweep_phase on resident data
template <int G, int MODE>
__device__ __forceinline__ void cycle_row(const TileArgs &a, const CycleCtx &x, int j, uint32_t sweep, const float2 nbeta,
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
    const float2 own = x.own[j * 32];
    auto neighbour = [&](int k) { return ldc_f2(x.ids[pos + k] + x.q8); };
    // the gathers first (the only remote reads of the row): up to kDB neighbours in registers
    float2 v[kDB];
#pragma unroll
    for (int u = 0; u < kDB; ++u) {
        v[u] = make_float2(0.f, 0.f);
        if (u < deg) v[u] = neighbour(u);
    }

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
    for (int u = 0; u < kDB; ++u)
        if (u < deg) acc.add(v[u], u);
    for (int k = kDB; k < dmax; k += 4) {    // rare: P(deg > 8) ~ 15 % at z = 6
        float2 t[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (k + u < deg) t[u] = neighbour(k + u);
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
        x.own[j * 32] = out;
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
                atomicAdd(x.sacc + x.q * 6, static_cast<unsigned long long>(__double2ll_rn(static_cast<double>(ex) * 524288.0)));
                atomicAdd(x.sacc + x.q * 6 + 3, static_cast<unsigned long long>(__double2ll_rn(static_cast<double>(ey) * 524288.0)));
            }
            iacc[1] += quant1(cx); iacc[2] += quant1(sx);
            iacc[4] += quant1(cy); iacc[5] += quant1(sy);
        }
    }
}

// the leader's conversion of a tallied sweep (sweep_finalize's arithmetic on resident data): slot r's fixed-point sums are
// the growth, since the last time this buffer was read, of the CTAs' running sums (collected through DSMEM; 64-bit
// wrap-around arithmetic is exact); E and M go to global memory (stores only), the accumulators stay in shared memory
struct CycleLeader {
    unsigned long long prev[2][64][3];      // running totals seen at the last read, per buffer and slot
    double accum[64][8];                    // the sample's accumulators by temperature (Eq. 13-16), resident
    int tos[64];                            // temp_of_slot
};

template <int G>
__device__ __forceinline__ void cycle_finalize(const TileArgs &a, CycleLeader &ld, uint32_t sacc_addr, int buf, int n_cta, int s,
                                               bool accumulate) {
    for (int r = threadIdx.x; r < 2 * G; r += blockDim.x) {
        unsigned long long tot[3] = {0ull, 0ull, 0ull};
        const uint32_t addr = sacc_addr + static_cast<uint32_t>(((buf * G + r / 2) * 6 + (r % 2) * 3) * 8);
        for (int c = 0; c < n_cta; ++c)
#pragma unroll
            for (int k = 0; k < 3; ++k) tot[k] += ld_cluster_u64(addr + k * 8, static_cast<uint32_t>(c));
        long long f[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            f[k] = static_cast<long long>(tot[k] - ld.prev[buf][r][k]);
            ld.prev[buf][r][k] = tot[k];
        }
        const double e = -static_cast<double>(f[0]) * kInvScaleE;
        const double mx = static_cast<double>(f[1]) * kInvScaleM;
        const double my = static_cast<double>(f[2]) * kInvScaleM;
        const size_t sr = static_cast<size_t>(s) * a.R + r;
        a.E_slot[sr] = e;
        a.M_slot[2 * sr] = mx;
        a.M_slot[2 * sr + 1] = my;
        if (accumulate) {
            double *o = ld.accum[ld.tos[r]];
            const double ux = mx / a.N, uy = my / a.N, m2 = ux * ux + uy * uy;
            o[0] += 1.0; o[1] += e; o[2] += e * e; o[3] += sqrt(m2); o[4] += m2; o[5] += m2 * m2;
            o[6] += ux; o[7] += uy;
        }
    }
}

template <int G, int ORDER>
__global__ void __launch_bounds__(kCycleWarps * 32, 512 / (kCycleWarps * 32)) k_cycle(const CycleArgs a) {
    constexpr int W = kCycleWarps;
    constexpr int SPW = 32 / G;
    extern __shared__ __align__(16) unsigned char s_raw[];
    __shared__ unsigned short s_jb[W][kCycleMaxQ + 1];      // per warp: first resident row of every colour class
    __shared__ int s_cp[kCycleMaxQ + 1];                       // first site of every colour class
    __shared__ int s_rb[kCycleMaxQ + 1][kCycleMaxCtas];        // rows of the classes before c owned by CTA b
    __shared__ unsigned long long s_acc[2][G][6];            // the CTA's running measured sums (exact integers), two buffers
    __shared__ CycleLeader s_ld;                             // used by the leader CTA only
    const TileArgs &t = a.t;

    CycleCtx x;
    x.s = t.s0 + blockIdx.y;
    x.lane = threadIdx.x & 31;
    x.sub = x.lane / G;
    x.q = x.lane % G;
    const int warp = threadIdx.x >> 5;
    x.lb = reinterpret_cast<float2 *>(t.theta) + static_cast<size_t>(x.s) * t.N * G + x.q;
    const size_t pool_bytes = cycle_pool_bytes(G, a.k_cap, a.id_cap);
    unsigned char *pool = s_raw + static_cast<size_t>(warp) * pool_bytes;
    x.own = reinterpret_cast<float2 *>(pool) + x.lane;
    int2 *meta = reinterpret_cast<int2 *>(pool + static_cast<size_t>(a.k_cap) * 256);
    uint32_t *ids = reinterpret_cast<uint32_t *>(pool + static_cast<size_t>(a.k_cap) * (256 + SPW * 8));
    x.meta = meta;
    x.ids = ids;
    x.q8 = static_cast<uint32_t>(x.q) * 8u;
    const uint32_t dyn_base = static_cast<uint32_t>(__cvta_generic_to_shared(s_raw));
    x.sacc = &s_acc[0][0][0];
    const uint32_t sacc_addr = static_cast<uint32_t>(__cvta_generic_to_shared(&s_acc[0][0][0]));
    const int n_cta = gridDim.x;
    const bool leader = blockIdx.x == 0;                 // cluster dims (C, 1, 1), grid (C, samples): rank = blockIdx.x

    // ---- once per launch: the sample moves into the cluster's shared memory.  CTA b owns rows [ceil(b n_c / C),
    // ceil((b+1) n_c / C)) of every colour class c (n_c rows): the sites of a class keep their lattice order (colour-major
    // numbering), so a CTA holds the same REGION of the lattice in every class and most neighbours of its sites are in
    // its own shared memory.  Inside the CTA its rows, numbered class after class (nu), go to warp nu mod W as that
    // warp's row nu div W -- closed forms, so a neighbour's location needs no table. ----
    if (threadIdx.x == 0) {
        const int32_t *cp = t.class_ptr + x.s * t.q_stride;
        for (int c = 0; c <= a.q_max; ++c) s_cp[c] = cp[c];
        for (int b = 0; b < n_cta; ++b) {
            int before = 0;
            for (int c = 0; c <= a.q_max; ++c) {
                s_rb[c][b] = before;                     // rows of the classes < c that CTA b owns
                if (c < a.q_max) {
                    const int n_rows = (cp[c + 1] - cp[c] + SPW - 1) / SPW;
                    before += cycle_first_row(b + 1, n_rows, n_cta) - cycle_first_row(b, n_rows, n_cta);
                }
            }
        }
    }
    for (int e = threadIdx.x; e < 2 * G * 6; e += blockDim.x) (&s_acc[0][0][0])[e] = 0ull;
    if (leader) {
        for (int e = threadIdx.x; e < 2 * 64 * 3; e += blockDim.x) (&s_ld.prev[0][0][0])[e] = 0ull;
        for (int e = threadIdx.x; e < 2 * G * 8; e += blockDim.x)
            s_ld.accum[e / 8][e % 8] = t.acc[(static_cast<size_t>(x.s) * t.R + e / 8) * 8 + e % 8];
        for (int r = threadIdx.x; r < 2 * G; r += blockDim.x) s_ld.tos[r] = t.temp_of_slot[static_cast<size_t>(x.s) * t.R + r];
    }
    __syncthreads();
    {
        const int2 *rec = t.rec + static_cast<size_t>(x.s) * t.N;
        int j = 0, n_ids = 0;
        for (int c = 0; c < a.q_max; ++c) {
            if (x.lane == 0) s_jb[warp][c] = static_cast<unsigned short>(j);
            const int cbeg = s_cp[c], cend = s_cp[c + 1];
            const int n_rows = (cend - cbeg + SPW - 1) / SPW;
            const int k_first = cycle_first_row(blockIdx.x, n_rows, n_cta), mine = cycle_first_row(blockIdx.x + 1, n_rows, n_cta) - k_first;
            for (int kk = (warp - s_rb[c][blockIdx.x] % W + W) % W; kk < mine; kk += W, ++j) {
                const int i = cbeg + (k_first + kk) * SPW + x.sub;
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
                for (int e = x.q; e < deg; e += G) {     // where neighbour n lives: class, row, owner warp and its row number
                    const int n = t.col_idx[rc.x + e];
                    int cn = 0;
                    while (cn + 1 < a.q_max && n >= s_cp[cn + 1]) ++cn;
                    const int kn = (n - s_cp[cn]) / SPW, sbn = (n - s_cp[cn]) % SPW;
                    const int nr = (s_cp[cn + 1] - s_cp[cn] + SPW - 1) / SPW;
                    const int bn = static_cast<int>(static_cast<long long>(kn) * n_cta / nr);      // the CTA whose range holds row kn
                    const int nu = s_rb[cn][bn] + kn - cycle_first_row(bn, nr, n_cta);
                    const uint32_t off = static_cast<uint32_t>((nu % W) * pool_bytes) + static_cast<uint32_t>((nu / W) * 256 + sbn * G * 8);
                    ids[pos + e] = bn == static_cast<int>(blockIdx.x) ? dyn_base + off : cluster_map(dyn_base + off, static_cast<uint32_t>(bn));
                }
                if (x.q == 0) meta[j * SPW + x.sub] = make_int2(valid ? i : -1, pos | (deg << 16) | (nlow << 24));
                x.own[j * 32] = valid ? x.lb[static_cast<unsigned long long>(static_cast<uint32_t>(i) * static_cast<uint32_t>(G))]
                                      : make_float2(0.f, 0.f);
                n_ids += total;
            }
        }
        if (x.lane == 0) s_jb[warp][a.q_max] = static_cast<unsigned short>(j);
    }
    __syncthreads();

    const uint32_t sweep0 = t.counters[0], round0 = t.counters[1];
    int iacc[6] = {0, 0, 0, 0, 0, 0};
    float2 nbeta = make_float2(0.f, 0.f), w = nbeta;     // this lane's -beta and proposal width: reloaded after every swap round
    bool reload = true;
    int tallied = 0;                                     // tallied sweeps so far: sweep n adds to buffer n % 2
    int finalize_pending = 0;                            // 1: convert the last tallied sweep's sums, 3: ... and accumulate them

    auto finalize_if_pending = [&]() {
        if (finalize_pending) {
            if (leader) cycle_finalize<G>(t, s_ld, sacc_addr, (tallied - 1) & 1, n_cta, x.s, (finalize_pending & 2) != 0);
            finalize_pending = 0;
        }
    };
    // one colour class: wait until the cluster has finished the previous class, update the warp's rows of the class.
    // The leader converts a finished sweep's sums right after the wait (all CTAs' sums are visible then).
    auto phase = [&](auto mode, int colour, uint32_t sweep) {
        constexpr int MODE = decltype(mode)::value;
        constexpr bool kMet = MODE == kModeMetropolis || MODE == kModeMetOr || MODE == kModeMetOrMeasure;
        const int j0 = s_jb[warp][colour], j1 = s_jb[warp][colour + 1];
        cluster_wait();
        finalize_if_pending();
        if constexpr (kMet) {
            if (reload) {      // first Metropolis class after a swap round: the leader's new beta / width per slot (global memory)
                const float2 b = __ldcg(reinterpret_cast<const float2 *>(t.beta_slot) + static_cast<size_t>(x.s) * G + x.q);
                nbeta = make_float2(-b.x, -b.y);
                w = __ldcg(reinterpret_cast<const float2 *>(t.w_slot) + static_cast<size_t>(x.s) * G + x.q);
                reload = false;
            }
        }
        for (int j = j0; j < j1; ++j) cycle_row<G, MODE>(t, x, j, sweep, nbeta, w, iacc);
    };
    // the sweep's E, Mx, My: per-lane partial sums -> the CTA's running sums in shared memory (exact 64-bit integer
    // atomics); the arrive that follows publishes them, the leader collects them after the next wait
    auto tally_done = [&](bool accumulate) {
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            long long v = iacc[c];
#pragma unroll
            for (int o = G; o < 32; o <<= 1) v += __shfl_xor_sync(kFull, v, o);      // the row's sites share the slot pair
            if (x.sub == 0 && v != 0) atomicAdd(x.sacc + x.q * 6 + c, static_cast<unsigned long long>(v));
            iacc[c] = 0;
        }
        tallied += 1;
        x.sacc = &s_acc[tallied & 1][0][0];              // the next tallied sweep adds to the other buffer
        finalize_pending = accumulate ? 3 : 1;
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
                    cluster_arrive_shared();
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
                        cluster_arrive_shared();
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
                    cluster_arrive_shared();
                }
            }
        }
        if (a.do_swap) {
            // end of the cycle: the leader converts the last sweep's sums (E per slot to global memory) and makes the swap
            // round there; the arrive that follows publishes the new beta / width per slot to the whole cluster
            cluster_wait();
            if (leader) {
                cycle_finalize<G>(t, s_ld, sacc_addr, (tallied - 1) & 1, n_cta, x.s, (finalize_pending & 2) != 0);
                __syncthreads();
                pt_swap_sample(a.sw, x.s, round0 + static_cast<uint32_t>(cyc));
                __syncthreads();
                for (int r = threadIdx.x; r < 2 * G; r += blockDim.x) s_ld.tos[r] = t.temp_of_slot[static_cast<size_t>(x.s) * t.R + r];
            }
            finalize_pending = 0;
            reload = true;
            cluster_arrive();
        }
    }
    cluster_wait();
    // ---- the launch ends: angles (and the leader's accumulators) go back to global memory ----
    for (int j = 0, nj = s_jb[warp][a.q_max]; j < nj; ++j) {
        const int2 m = x.meta[j * SPW + x.sub];
        if (m.x >= 0) x.lb[static_cast<unsigned long long>(static_cast<uint32_t>(m.x) * static_cast<uint32_t>(G))] = x.own[j * 32];
    }
    if (leader) {
        __syncthreads();
        for (int e = threadIdx.x; e < 2 * G * 8; e += blockDim.x)
            t.acc[(static_cast<size_t>(x.s) * t.R + e / 8) * 8 + e % 8] = s_ld.accum[e / 8][e % 8];
    }
    // (no CTA reads another one's shared memory after the last wait: every remote read precedes its reader's arrive)
}

}  // namespace xy
