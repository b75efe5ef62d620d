// xy_sweep.cuh -- the colour-class kernel k_phase<G, CB, MODE, W>: Metropolis and/or over-relaxation update of one
// colour class (optionally with the E / M measurement as a by-product), or the stand-alone E / M reduction over all
// sites, for one group of samples.
//
// Work layout: theta[S][N][R] fp32, replica fastest.  A lane owns TWO adjacent slots (one float2, one Philox4x32-10
// call per site: words (x0,x1) feed the even slot, (x2,x3) the odd one), G = R/2 lanes cover a site (G = 32 and
// column blocks of 64 slots when R % 64 == 0) and a warp works on SPW = 32/G sites at once ("row").  At R = 64 one
// neighbour gather is one fully used 256-byte request.  A warp owns a contiguous, cost-balanced share of the colour
// class and walks it in chunks of <= 32 sites: one coalesced load of the chunk's rec[], the chunk's neighbour ids
// (one contiguous CSR run) staged in the warp's slice of shared memory, pre-scaled by the site stride.  Same-colour
// sites share no bond, so the gathers of row t+1 never read what row t stores: they are issued BEFORE
// row t is computed, as cp.async (LDGSTS) copies of the lane's own 8 bytes into a per-warp ring in shared memory --
// in-flight data costs no registers (64 per thread and 32 warps per SM for the update modes, without spills; 80
// registers and 24 warps for the interleaved mode that also measures, 72 registers and 28 warps for the over-relaxation
// that also measures), each lane reads back only what it copied itself
// (cp.async.wait_group, no cross-lane synchronisation), and the Philox / sin / exp work of row t covers the latency
// of row t+1.  When SPW > 1 the sites of a row have different degrees: the loops run to the row maximum and lanes
// whose site has fewer neighbours are predicated off (no memory request is made for them).
//
// Modes: 0 Metropolis, 1 over-relaxation, 2 measure, 3 over-relaxation + measurement by-product, 4 Metropolis then
// over-relaxation of the same site from one gather (interleaved order, xy_set_order), 5 = 4 + measurement by-product.
//
// The launches of a PT cycle are captured in a CUDA graph with PROGRAMMATIC DEPENDENT LAUNCH edges (see k_phase).
// Small samples run whole cycles in one launch instead: one thread-block cluster per sample with the hardware cluster
// barrier between the colour classes (k_cycle, xy_cycle.cuh), built from the same sweep_prep / sweep_phase pieces.
//
// PAPER.md:444,:454 (coloured single-spin Metropolis), :460 (over-relaxation, ref 66), :167-181 (E, m),
// :460-472 (parallel tempering); readings R5-R11, R20 in DESIGN.md.
#pragma once
#include "xy_kernels.cuh"

namespace xy {

constexpr int kDB = 8;            // pipelined gathers per site
constexpr int kDepth = 2;         // ring slots per warp (rows in flight)
constexpr int kStageCap = 256;    // staged neighbour ids per warp and chunk (ints)
// k_phase comes in two CTA shapes with the same 32 resident warps per SM (64 registers): W = 32 warps (one CTA per SM)
// for large colour classes, W = 8 (four CTAs per SM) for small ones.  Measured: the SM's warp scheduler
// favours older CTAs, so four co-resident CTAs finish 2-3 us apart and the SM idles in the tail; the warps of ONE CTA
// progress evenly (+8 % on config 4).  Small classes prefer the finer CTA granularity.
constexpr int kWarpsBig = 32, kWarpsSmall = 8;
constexpr int kSmPerWarpSlots = 32;                    // resident warps per SM the register / shared budget is sized for

// fixed-point scales of the measure reduction (exact, order-independent integer sums; see quant8 / quant1)
constexpr double kInvScaleE = 1.0 / 524288.0;      // 2^-19
constexpr double kInvScaleM = 1.0 / 4194304.0;     // 2^-22

// per warp: ring[kDepth][kDB + 1][32] float2 (row kDB = the site's own angle) + staged ids
struct __align__(16) SweepWarp {
    float2 ring[kDepth][kDB + 1][32];
    uint32_t idx[kStageCap];
};
constexpr size_t sweep_smem(int warps) { return sizeof(SweepWarp) * warps; }     // dynamic shared memory of a k_phase CTA
static_assert(sweep_smem(kSmPerWarpSlots) <= 227 * 1024 - 4 * 1024, "shared memory per SM");
static_assert(sizeof(SweepWarp) >= sizeof(long long) * 32 * 6, "measure reduction reuses the ring");

// ---- packed fp32x2 helpers (IEEE rn per component: bit-identical to the scalar operations) ----------
__device__ __forceinline__ float2 add2(const float2 a, const float2 b) {
    float2 r;
    asm("{ .reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; add.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc; }"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 sub2(const float2 a, const float2 b) { return add2(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ float2 mul2(const float2 a, const float2 b) {
    float2 r;
    asm("{ .reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mul.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc; }"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}

// as_float((x >> 9) | 0x3f800000) = 1 + k 2^-23, k = x >> 9
__device__ __forceinline__ float mant12(uint32_t x) { return __uint_as_float((x >> 9) | 0x3f800000u); }

// float -> fixed point by the magic-number add (one FADD.rn + one IADD, deterministic):
//   |x| <= 8:  x + 24 lies in [16, 32], ulp 2^-19, so bits(x + 24) - bits(24) = rn(x 2^19)
//   |x| <= 1:  x + 3  lies in [2, 4],   ulp 2^-22, so bits(x + 3)  - bits(3)  = rn(x 2^22)
__device__ __forceinline__ int quant8(float x) { return __float_as_int(__fadd_rn(x, 24.0f)) - 0x41C00000; }
__device__ __forceinline__ int quant1(float x) { return __float_as_int(__fadd_rn(x, 3.0f)) - 0x40400000; }
//   |x| <= 32: x + 96 lies in [64, 128], ulp 2^-17, so bits(x + 96) - bits(96) = rn(x 2^17)
__device__ __forceinline__ int quant32(float x) { return __float_as_int(__fadd_rn(x, 96.0f)) - 0x42C00000; }

// ---- per-lane state of one site (two slots) ----------------------------------------------------------
// add(t, k): t = the angles of the site's k-th neighbour (CSR order) in the lane's two slots
template <int MODE> struct PairAcc;
template <> struct PairAcc<kModeMetropolis> {
    float2 mid, s = make_float2(0.f, 0.f);
    __device__ __forceinline__ void add(const float2 t, int) {
        const float2 d = sub2(mid, t);
        s = add2(s, make_float2(__sinf(d.x), __sinf(d.y)));
    }
};
template <> struct PairAcc<kModeOverrelax> {
    float2 hx = make_float2(0.f, 0.f), hy = make_float2(0.f, 0.f);   // hx = (h_x of slot .x, h_x of slot .y)
    __device__ __forceinline__ void add(const float2 t, int) {
        float sx, cx, sy, cy;
        __sincosf(t.x, &sx, &cx);
        __sincosf(t.y, &sy, &cy);
        hx = add2(hx, make_float2(cx, cy));
        hy = add2(hy, make_float2(sx, sy));
    }
};
// measure: l = sum over the LOWER neighbours j < i (the head of the ascending list: every bond is counted once, at
// its upper end) of (cos th_j, sin th_j); the bond energy of the site is then cos th_i l_x + sin th_i l_y
// (site_energy_fixed).  Only lower neighbours are gathered, so every add() is a lower one.
template <> struct PairAcc<kModeMeasure> {
    float2 lx = make_float2(0.f, 0.f), ly = make_float2(0.f, 0.f);
    __device__ __forceinline__ void add(const float2 t, int) {
        float sx, cx, sy, cy;
        __sincosf(t.x, &sx, &cx);
        __sincosf(t.y, &sy, &cy);
        lx = add2(lx, make_float2(cx, cy));
        ly = add2(ly, make_float2(sx, sy));
    }
};
// over-relaxation with the measurement as a by-product: the local field h needs (cos th_j, sin th_j) of every
// neighbour anyway; the partial field l of the lower neighbours is a prefix of that sum -- the same terms in the same
// order that the measure kernel adds, so both give bit-identical energies.  After the class's update th_i and all its lower neighbours are
// final for this sweep (colour-major numbering: j < i has a lower or equal colour, and same-colour sites share no bond).
template <> struct PairAcc<kModeOrMeasure> {
    float2 hx = make_float2(0.f, 0.f), hy = make_float2(0.f, 0.f), lx = make_float2(0.f, 0.f), ly = make_float2(0.f, 0.f);
    int nlow = 0;
    __device__ __forceinline__ void add(const float2 t, int k) {
        float sx, cx, sy, cy;
        __sincosf(t.x, &sx, &cx);
        __sincosf(t.y, &sy, &cy);
        hx = add2(hx, make_float2(cx, cy));
        hy = add2(hy, make_float2(sx, sy));
        if (k == nlow - 1) {     // the lower neighbours are the head of the list: l is h's partial sum after the last of them
            lx = hx;
            ly = hy;
        }
    }
};

// interleaved order (xy_set_order): Metropolis and then over-relaxation of the SAME site from
// ONE gather.  Same-colour sites share no bond, so the neighbours do not change between the two updates, and the local
// field h = sum_j (cos th_j, sin th_j) serves both: sum_j sin(mid - th_j) = sin(mid) h_x - cos(mid) h_y.
template <> struct PairAcc<kModeMetOr> : PairAcc<kModeOverrelax> {};
template <> struct PairAcc<kModeMetOrMeasure> : PairAcc<kModeOrMeasure> {};

// fixed-point (scale 2^19) bond energy of one slot of a site: -E_i = cos th_i l_x + sin th_i l_y, |.| <= nlow.
// Explicit fma/mul so that the measure kernel and the fused over-relaxation kernel round identically.
__device__ __forceinline__ float site_energy(float c, float s, float lx, float ly) {
    return __fmaf_rn(c, lx, __fmul_rn(s, ly));
}
// per-lane description of the site a lane works on in the current row (warp-uniform when SPW == 1)
struct RowSite { int i, deg, pos, nlow; bool valid; };

// direct gather of the neighbour with pre-scaled id `sid` (float2 units), L2 only: one IMAD.WIDE.U32 + one LDG.64
__device__ __forceinline__ float2 sweep_ld(const float2 *lb, uint32_t sid) {
    return __ldcg(lb + static_cast<unsigned long long>(sid));
}

// issue D async gathers back to back; UNI: every lane has at least D neighbours (nothing predicated off)
template <int D, bool UNI>
__device__ __forceinline__ void sweep_issue_n(uint32_t row0, const float2 *lb, const uint32_t *sidx, int pos, int deg) {
    uint32_t sid[D];
#pragma unroll
    for (int u = 0; u < D; ++u) {      // all id loads first: LDS -> LDGSTS hazards are paid once
        sid[u] = 0u;
        if (UNI || u < deg) sid[u] = sidx[pos + u];
    }
#pragma unroll
    for (int u = 0; u < D; ++u)
        if (UNI || u < deg) cp_async8(row0 + u * 256u, lb + static_cast<unsigned long long>(sid[u]));
}

// row0 = shared address of this lane's 8 bytes in row 0 of the ring slot; dmax = warp maximum of deg
template <bool UNI>
__device__ __forceinline__ void sweep_issue(uint32_t row0, const float2 *lb, const uint32_t *sidx, int pos, int deg, int dmax) {
    switch (dmax < kDB ? dmax : kDB) {
        case 8: sweep_issue_n<8, UNI>(row0, lb, sidx, pos, deg); break;
        case 7: sweep_issue_n<7, UNI>(row0, lb, sidx, pos, deg); break;
        case 6: sweep_issue_n<6, UNI>(row0, lb, sidx, pos, deg); break;
        case 5: sweep_issue_n<5, UNI>(row0, lb, sidx, pos, deg); break;
        case 4: sweep_issue_n<4, UNI>(row0, lb, sidx, pos, deg); break;
        case 3: sweep_issue_n<3, UNI>(row0, lb, sidx, pos, deg); break;
        case 2: sweep_issue_n<2, UNI>(row0, lb, sidx, pos, deg); break;
        case 1: sweep_issue_n<1, UNI>(row0, lb, sidx, pos, deg); break;
        default: break;
    }
}

// batches of <= 4 LDS.64 then their arithmetic (8 at once would cost 16 registers at the kernel's pressure peak)
template <int D, bool UNI, typename ACC>
__device__ __forceinline__ void sweep_consume_n(ACC &acc, const float2 *row0, int deg) {
#pragma unroll
    for (int b = 0; b < D; b += 4) {
        float2 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (b + u < D) v[u] = row0[(b + u) * 32];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (b + u < D && (UNI || b + u < deg)) acc.add(v[u], b + u);
    }
}

// row0 = pointer to this lane's float2 in row 0 of the ring slot: the first min(deg, kDB) neighbours
template <bool UNI, typename ACC>
__device__ __forceinline__ void sweep_consume(ACC &acc, const float2 *row0, int deg, int dmax) {
    switch (dmax < kDB ? dmax : kDB) {
        case 8: sweep_consume_n<8, UNI>(acc, row0, deg); break;
        case 7: sweep_consume_n<7, UNI>(acc, row0, deg); break;
        case 6: sweep_consume_n<6, UNI>(acc, row0, deg); break;
        case 5: sweep_consume_n<5, UNI>(acc, row0, deg); break;
        case 4: sweep_consume_n<4, UNI>(acc, row0, deg); break;
        case 3: sweep_consume_n<3, UNI>(acc, row0, deg); break;
        case 2: sweep_consume_n<2, UNI>(acc, row0, deg); break;
        case 1: sweep_consume_n<1, UNI>(acc, row0, deg); break;
        default: break;
    }
}

// ---- arguments: the shared TileArgs plus the share table ---------------------------------------------------------
struct SweepArgs {
    TileArgs t;
    const int4 *part;              // [S][q_stride][nw] per warp {first site, end site, first col_idx entry and number of
                                   // staged ids of the share's first chunk}: cost-balanced shares (colour q_max = the
                                   // measure pass over all sites), nw = warps per sample and column block; nullptr = equal shares
};

// per-thread constants of a launch
struct SweepCtx {
    float2 *lb;                 // this lane's column of the sample: theta2 + s*N*R2 + q
    const int2 *rec;            // rec of the sample
    uint32_t *sidx;             // the warp's staged ids
    const float2 *ring_l;       // this lane's column of the warp's ring (generic pointer)
    uint32_t ring_s;            // same, shared-space address
    int s, lane, warp, sub, q;
    long long *fx;              // the fixed-point sums the measuring modes add to ([S][R][3]; k_cycle alternates two buffers)
};

// what a warp stages BEFORE it waits for the preceding launch (graph data only, never theta): its share
// [i0, w1) of the colour class, the rec[] of the share's first chunk, and that chunk's neighbour ids in shared memory
struct PhasePrep { int i0, w1; int2 rc; };

// leading sites of a chunk whose neighbour ids fit the staging slice; start0 = first col_idx entry of the chunk,
// endl = end of this lane's list relative to start0
__device__ __forceinline__ int chunk_fit(const int2 rc, int lane, int nsite, int &start0, int &endl) {
    start0 = __shfl_sync(kFull, rc.x, 0);
    endl = rc.x + (rc.y & 0xffff) - start0;
    const unsigned fits = __ballot_sync(kFull, lane < nsite && endl <= kStageCap);
    return fits == kFull ? 32 : __ffs(~fits) - 1;
}

// stage the chunk's ids (pre-scaled by the site stride): 4 loads in flight per lane
__device__ __forceinline__ void chunk_stage(const int32_t *gidx, uint32_t *sidx, int lane, int n_run, uint32_t R2) {
    for (int p0 = 0; p0 < n_run; p0 += 128) {
        int32_t g[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (p0 + u * 32 + lane < n_run) g[u] = gidx[p0 + u * 32 + lane];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (p0 + u * 32 + lane < n_run) sidx[p0 + u * 32 + lane] = static_cast<uint32_t>(g[u]) * R2;
    }
}

// nw warps share the class, this warp is number gw of them (nw = gridDim.x * W, gw = blockIdx.x * W + warp); use_part:
// take the cost-balanced share table when there is one
template <int G, int CB>
__device__ __forceinline__ PhasePrep sweep_prep(const SweepArgs &sa, const SweepCtx &x, int mode, int colour, int nw, int gw,
                                                bool use_part) {
    constexpr int SPW = 32 / G;
    const TileArgs &a = sa.t;
    const uint32_t R2 = CB ? static_cast<uint32_t>(G) : static_cast<uint32_t>(a.R >> 1);
    PhasePrep P;
    P.rc = make_int2(0, 0);
    const int cidx = mode == kModeMeasure ? a.q_stride - 1 : colour;
    if (use_part && sa.part) {      // cost-balanced shares (host-computed: cost = const + degree)
        const int4 e = __ldg(sa.part + (static_cast<size_t>(x.s) * a.q_stride + cidx) * nw + gw);
        P.i0 = e.x; P.w1 = e.y;
        if (P.i0 < P.w1) {      // rec[] and the ids of the first chunk in parallel: two dependent latencies, not three
            if (x.lane < min(32, P.w1 - P.i0)) P.rc = x.rec[P.i0 + x.lane];
            if (e.w > 0) chunk_stage(a.col_idx + e.z, x.sidx, x.lane, e.w, R2);
        }
        return P;
    } else {            // contiguous equal shares (whole rows)
        int cbeg = 0, cend = a.N;
        if (mode != kModeMeasure) {
            cbeg = a.class_ptr[x.s * a.q_stride + colour];
            cend = a.class_ptr[x.s * a.q_stride + colour + 1];
        }
        const int per = ((cend - cbeg + nw - 1) / nw + SPW - 1) / SPW * SPW;
        P.i0 = min(cend, cbeg + gw * per); P.w1 = min(cend, P.i0 + per);
    }
    if (P.i0 < P.w1) {
        const int nsite = min(32, P.w1 - P.i0);
        if (x.lane < nsite) P.rc = x.rec[P.i0 + x.lane];
        int start0, endl;
        const int msite = chunk_fit(P.rc, x.lane, nsite, start0, endl);
        if (msite > 0) chunk_stage(a.col_idx + start0, x.sidx, x.lane, __shfl_sync(kFull, endl, msite - 1), R2);
    }
    return P;
}

// ---- one phase: MODE 0 Metropolis / 1 over-relaxation / 3 over-relaxation + measure by-product on a colour class,
// 2 measure on all sites ----
// G lanes per site; CB = 1: the site stride R/2 equals G (known at compile time), CB = 0: G = 32, R a multiple of 64
// larger than 64 (blockIdx.z = block of 64 slots).  P: the share and its first chunk as staged by sweep_prep (the
// staged ids are visible: a __syncwarp separates the two).  iacc: measure modes only, 32-bit fixed-point partial sums
// (E, Mx, My) of the .x slot, then of the .y slot.
template <int G, int CB, int MODE>
__device__ __forceinline__ void sweep_phase(const TileArgs &a, const SweepCtx &x, const PhasePrep &P, uint32_t sweep,
                                            int (&iacc)[6]) {
    constexpr int SPW = 32 / G;
    constexpr bool UNI = SPW == 1;
    const uint32_t R2 = CB ? static_cast<uint32_t>(G) : static_cast<uint32_t>(a.R >> 1);
    constexpr uint32_t kSlotBytes = (kDB + 1) * 32 * sizeof(float2);
    constexpr int kSlotElems = (kDB + 1) * 32;
    const int s = x.s, lane = x.lane, sub = x.sub;
    float2 *lb = x.lb;
    const int2 *__restrict__ rec = x.rec;
    uint32_t *sidx = x.sidx;
    const int w1 = P.w1;
    if (P.i0 >= w1) return;

    float2 nbeta = make_float2(0.f, 0.f), w = make_float2(0.f, 0.f);
    uint32_t c2 = 0;
    constexpr bool kMet = MODE == kModeMetropolis || MODE == kModeMetOr || MODE == kModeMetOrMeasure;
    constexpr bool kFusedMetOr = MODE == kModeMetOr || MODE == kModeMetOrMeasure;
    constexpr bool kTally = MODE == kModeMeasure || MODE == kModeOrMeasure || MODE == kModeMetOrMeasure;
    if constexpr (kMet) {
        const float2 b = __ldcg(reinterpret_cast<const float2 *>(a.beta_slot) + static_cast<size_t>(s) * R2 + x.q);
        nbeta = make_float2(-b.x, -b.y);
        w = __ldcg(reinterpret_cast<const float2 *>(a.w_slot) + static_cast<size_t>(s) * R2 + x.q);
        c2 = ((a.sample_base + static_cast<uint32_t>(s)) << 16) | static_cast<uint32_t>(x.q);
    }

    // Metropolis proposal of site i (both slots of the lane): th' = th + w (u1 - 1/2), half = (th' - th)/2
    auto begin = [&](int i, int nlow, const float2 own, PairAcc<MODE> &acc, float2 &thp, float2 &u2) {
        if constexpr (kMet) {
            uint32_t r[4];
            philox4x32_10(static_cast<uint32_t>(i), sweep, c2, kDomMetropolis, a.keys, r);
            // u = (k + 1/2) 2^-23 with k = x >> 9 (R11), every step exact:
            //   u1 - 1/2 = ((1 + k 2^-23) - 3/2) + 2^-24,   u2 = (1 + k 2^-23) - (1 - 2^-24)
            const float2 u1mh = add2(add2(make_float2(mant12(r[0]), mant12(r[2])), make_float2(-1.5f, -1.5f)),
                                     make_float2(5.9604644775390625e-08f, 5.9604644775390625e-08f));
            u2 = add2(make_float2(mant12(r[1]), mant12(r[3])), make_float2(-0.99999994f, -0.99999994f));
            // R5: delta = fp32(w * (u1 - 1/2)), th' = fp32(th + delta): two roundings.  Scalar mul.rn / add.rn on purpose:
            // ptxas contracts mul.rn.f32x2 + add.rn.f32x2 into one FFMA2 (single rounding, 1 ulp off in 11 % of the moves)
            thp = make_float2(__fadd_rn(own.x, __fmul_rn(w.x, u1mh.x)), __fadd_rn(own.y, __fmul_rn(w.y, u1mh.y)));
            if constexpr (MODE == kModeMetropolis) acc.mid = add2(own, mul2(sub2(thp, own), make_float2(0.5f, 0.5f)));
        }
        if constexpr (MODE == kModeOrMeasure || MODE == kModeMetOrMeasure) acc.nlow = nlow;
    };
    // measure by-product of one site: fixed-point bond energy (lower neighbours) and magnetisation of both slots
    // The per-lane partial sums are 32-bit.  A site adds at most 2^22 per quantity (one "unit"), or 2^24 to the energy
    // when it has 9..32 lower neighbours (coarser quantiser, 4 units); the partial sums are flushed to the 64-bit sums
    // in global memory before 2^31 can be reached (rarely: same-address atomics are slow).  A site with more than 32
    // lower neighbours goes to the 64-bit sum directly.
    auto fx_lane = [&]() {      // this lane's six 64-bit sums (recomputed where needed: cold code, no live registers)
        return reinterpret_cast<unsigned long long *>(x.fx) + (static_cast<size_t>(x.s) * a.R + 2 * x.q) * 3;
    };
    int units = 0;
    auto tally = [&](const float2 th, const float2 lx, const float2 ly, int nlow) {
        float sx, cx, sy, cy;
        __sincosf(th.x, &sx, &cx);
        __sincosf(th.y, &sy, &cy);
        const float ex = site_energy(cx, sx, lx.x, ly.x), ey = site_energy(cy, sy, lx.y, ly.y);
        units += 1;
        if (nlow <= 8) {
            iacc[0] += quant8(ex);
            iacc[3] += quant8(ey);
        } else if (nlow <= 32) {
            iacc[0] += quant32(ex) << 2;
            iacc[3] += quant32(ey) << 2;
            units += 3;
        } else {
            atomicAdd(fx_lane(), static_cast<unsigned long long>(__double2ll_rn(static_cast<double>(ex) * 524288.0)));
            atomicAdd(fx_lane() + 3, static_cast<unsigned long long>(__double2ll_rn(static_cast<double>(ey) * 524288.0)));
        }
        iacc[1] += quant1(cx); iacc[2] += quant1(sx);
        iacc[4] += quant1(cy); iacc[5] += quant1(sy);
    };
    auto flush_partial = [&]() {
        unsigned long long *fxl = fx_lane();
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            atomicAdd(fxl + c, static_cast<unsigned long long>(static_cast<long long>(iacc[c])));
            iacc[c] = 0;
        }
    };

    auto finish = [&](int i, int nlow, bool valid, const float2 own, PairAcc<MODE> &acc, const float2 thp, const float2 u2) {
        if constexpr (MODE == kModeMetropolis) {
            // dE = 2 sin((th'-th)/2) sum_j sin((th'+th)/2 - th_j)
            const float2 half = mul2(sub2(thp, own), make_float2(0.5f, 0.5f));      // recomputed: two registers fewer across the gather
            const float2 sh = make_float2(__sinf(half.x), __sinf(half.y));
            const float2 arg = mul2(nbeta, mul2(add2(sh, sh), acc.s));
            float2 out;
            out.x = metropolis_select(own.x, thp.x, u2.x, __expf(arg.x));
            out.y = metropolis_select(own.y, thp.y, u2.y, __expf(arg.y));
            if (UNI || valid) lb[static_cast<unsigned long long>(static_cast<uint32_t>(i) * R2)] = out;
        } else if constexpr (MODE == kModeOverrelax) {
            float2 out;
            out.x = overrelax_finish(own.x, acc.hx.x, acc.hy.x);
            out.y = overrelax_finish(own.y, acc.hx.y, acc.hy.y);
            if (UNI || valid) lb[static_cast<unsigned long long>(static_cast<uint32_t>(i) * R2)] = out;
        } else if constexpr (kFusedMetOr) {
            // Metropolis from the local field: dE = 2 sin((th'-th)/2) (sin(mid) h_x - cos(mid) h_y), then the
            // over-relaxation of the (possibly moved) spin about the same h
            const float2 half = mul2(sub2(thp, own), make_float2(0.5f, 0.5f));
            const float2 mid = add2(own, half);
            float smx, cmx, smy, cmy;
            __sincosf(mid.x, &smx, &cmx);
            __sincosf(mid.y, &smy, &cmy);
            const float2 ss = make_float2(__fmaf_rn(smx, acc.hx.x, -__fmul_rn(cmx, acc.hy.x)),
                                          __fmaf_rn(smy, acc.hx.y, -__fmul_rn(cmy, acc.hy.y)));
            const float2 sh = make_float2(__sinf(half.x), __sinf(half.y));
            const float2 arg = mul2(nbeta, mul2(add2(sh, sh), ss));
            float2 out;
            out.x = overrelax_finish(metropolis_select(own.x, thp.x, u2.x, __expf(arg.x)), acc.hx.x, acc.hy.x);
            out.y = overrelax_finish(metropolis_select(own.y, thp.y, u2.y, __expf(arg.y)), acc.hx.y, acc.hy.y);
            if (UNI || valid) {
                lb[static_cast<unsigned long long>(static_cast<uint32_t>(i) * R2)] = out;
                if constexpr (MODE == kModeMetOrMeasure) tally(out, acc.lx, acc.ly, nlow);
            }
        } else if constexpr (MODE == kModeOrMeasure) {
            float2 out;
            out.x = overrelax_finish(own.x, acc.hx.x, acc.hy.x);
            out.y = overrelax_finish(own.y, acc.hx.y, acc.hy.y);
            if (UNI || valid) {
                lb[static_cast<unsigned long long>(static_cast<uint32_t>(i) * R2)] = out;
                tally(out, acc.lx, acc.ly, nlow);
            }
        } else {
            if (UNI || valid) tally(own, acc.lx, acc.ly, nlow);
        }
    };
    // neighbours beyond the pipelined kDB: direct loads in groups of 4 (rare: P(deg > 8) ~ 15 % at z = 6)
    auto tail = [&](PairAcc<MODE> &acc, int pos, int deg, int dmax) {
        for (int k = kDB; k < dmax; k += 4) {
            float2 t[4];
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (k + u < deg) t[u] = sweep_ld(lb, sidx[pos + k + u]);
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (k + u < deg) acc.add(t[u], k + u);
        }
    };

    bool staged = true;      // the first chunk comes from sweep_prep
    int2 rc = P.rc;
    for (int i0 = P.i0; i0 < w1;) {
        // ---- chunk: the longest prefix of <= 32 sites whose neighbour ids fit the staging slice ----
        const int nsite = min(32, w1 - i0);
        if (!staged) {
            rc = make_int2(0, 0);
            if (lane < nsite) rc = rec[i0 + lane];
        }
        int start0, endl;
        const int msite = chunk_fit(rc, lane, nsite, start0, endl);

        if (msite == 0) {
            // a single site with more neighbours than the staging slice: lane group 0 walks its ids in blocks
            const int ry = __shfl_sync(kFull, rc.y, 0);
            int deg = ry & 0xffff;
            const int nlow = static_cast<int>(static_cast<uint32_t>(ry) >> 16);
            if constexpr (MODE == kModeMeasure) deg = nlow;      // lower neighbours only: the head of the list
            const int32_t *gidx = a.col_idx + start0;
            const bool valid = UNI || sub == 0;
            float2 own = make_float2(0.f, 0.f);
            if (valid) own = __ldcg(lb + static_cast<unsigned long long>(static_cast<uint32_t>(i0) * R2));
            float2 thp = make_float2(0.f, 0.f), u2 = thp;
            PairAcc<MODE> acc;
            begin(i0, nlow, own, acc, thp, u2);
            for (int k0 = 0; k0 < deg; k0 += kStageCap) {
                const int nb = min(kStageCap, deg - k0);
                __syncwarp();
                for (int p = lane; p < nb; p += 32) sidx[p] = static_cast<uint32_t>(gidx[k0 + p]) * R2;
                __syncwarp();
                for (int k = 0; k < nb; k += 4) {
                    float2 t[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        if (k + u < nb && valid) t[u] = sweep_ld(lb, sidx[k + u]);
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        if (k + u < nb && valid) acc.add(t[u], k0 + k + u);
                }
            }
            finish(i0, nlow, valid, own, acc, thp, u2);
            __syncwarp();
            i0 += 1;
            staged = false;
            if constexpr (kTally) {
                if (units >= 320 && i0 < w1) {      // a run of hub sites must not overflow the 32-bit partial sums either
                    flush_partial();
                    units = 0;
                }
            }
            continue;
        }

        if (!staged) {
            chunk_stage(a.col_idx + start0, sidx, lane, __shfl_sync(kFull, endl, msite - 1), R2);
            __syncwarp();
        }
        staged = false;

        rc.x -= start0;      // list starts relative to the staged run from here on (one register fewer in the row loop)
        auto site_of = [&](int t) {
            const int m = t * SPW + sub;
            const int ry = __shfl_sync(kFull, rc.y, m & 31), rx = __shfl_sync(kFull, rc.x, m & 31);
            RowSite st;
            st.valid = UNI || m < msite;
            st.i = i0 + m;
            st.deg = st.valid ? (ry & 0xffff) : 0;
            st.pos = rx;
            st.nlow = st.valid ? static_cast<int>(static_cast<uint32_t>(ry) >> 16) : 0;
            if constexpr (MODE == kModeMeasure) st.deg = st.nlow;   // bonds counted once: neighbours j < i are the head of the list
            return st;
        };
        auto row_max = [&](int deg) { return UNI ? deg : static_cast<int>(__reduce_max_sync(kFull, static_cast<unsigned>(deg))); };
        // async copies of the row (own angle -> ring row kDB, first kDB neighbours -> rows 0..) into ring slot `slot`
        auto issue = [&](const RowSite st, int dmax, int slot) {
            const uint32_t row0 = x.ring_s + static_cast<uint32_t>(slot) * kSlotBytes;
            if (st.valid) cp_async8(row0 + kDB * 256u, lb + static_cast<unsigned long long>(static_cast<uint32_t>(st.i) * R2));
            sweep_issue<UNI>(row0, lb, sidx, st.pos, st.deg, dmax);
            cp_async_commit();
        };

        // software pipeline over the chunk: the copies of row t+1 fly while row t is computed.  The row's site is
        // re-derived from rc (two shuffles) rather than carried across the iteration: registers matter more here.
        {
            const RowSite first = site_of(0);
            issue(first, row_max(first.deg), 0);
        }
        for (int t = 0; t * SPW < msite; ++t) {
            if ((t + 1) * SPW < msite) {
                const RowSite nxt = site_of(t + 1);
                issue(nxt, row_max(nxt.deg), (t + 1) & 1);
                cp_async_wait<1>();
            } else {
                cp_async_wait<0>();
            }
            const RowSite cur = site_of(t);
            const int cmax = row_max(cur.deg);
            const float2 *row0 = x.ring_l + (t & 1) * kSlotElems;
            float2 own = make_float2(0.f, 0.f);
            if (cur.valid) own = row0[kDB * 32];
            float2 thp = make_float2(0.f, 0.f), u2 = thp;
            PairAcc<MODE> acc;
            begin(cur.i, cur.nlow, own, acc, thp, u2);
            sweep_consume<UNI>(acc, row0, cur.deg, cmax);
            if (cmax > kDB) tail(acc, cur.pos, cur.deg, cmax);
            finish(cur.i, cur.nlow, cur.valid, own, acc, thp, u2);
        }
        __syncwarp();
        i0 += msite;
        if constexpr (kTally) {
            if (units >= 320 && i0 < w1) {      // a chunk adds at most 128 units: the partial sums stay below 448 * 2^22 < 2^31
                flush_partial();
                units = 0;
            }
        }
    }
}

// last CTA of a sample in a measure launch: fixed-point sums -> E, M per slot, optional accumulation under the
// slot's temperature (Eq. 13-16); leaves fx zeroed for the next measure launch
__device__ __forceinline__ void sweep_finalize(const TileArgs &a, long long *fx, int s, bool accumulate) {
    for (int r = threadIdx.x; r < a.R; r += blockDim.x) {
        long long *f = fx + (static_cast<size_t>(s) * a.R + r) * 3;
        const double e = -static_cast<double>(__ldcg(f)) * kInvScaleE;
        const double mx = static_cast<double>(__ldcg(f + 1)) * kInvScaleM;
        const double my = static_cast<double>(__ldcg(f + 2)) * kInvScaleM;
        f[0] = 0; f[1] = 0; f[2] = 0;
        const size_t sr = static_cast<size_t>(s) * a.R + r;
        a.E_slot[sr] = e;
        a.M_slot[2 * sr] = mx;
        a.M_slot[2 * sr + 1] = my;
        if (accumulate) {
            double *o = a.acc + (static_cast<size_t>(s) * a.R + __ldcg(a.temp_of_slot + sr)) * 8;
            const double ux = mx / a.N, uy = my / a.N, m2 = ux * ux + uy * uy;
            o[0] += 1.0; o[1] += e; o[2] += e * e; o[3] += sqrt(m2); o[4] += m2; o[5] += m2 * m2;
            o[6] += ux; o[7] += uy;
        }
    }
}

// the CTA's per-lane fixed-point partial sums -> one 64-bit atomic per (slot, quantity) and CTA; reuses the warps' ring
// slices as scratch, so all warps of the CTA must have left sweep_phase (block-wide barriers inside)
template <int G, int W>
__device__ __forceinline__ void sweep_reduce_to_fx(const TileArgs &a, const SweepCtx &x, const int (&iacc)[6], SweepWarp *s_w) {
    constexpr int SPW = 32 / G;
    __syncthreads();
    long long *s_red = reinterpret_cast<long long *>(&s_w[0]);
#pragma unroll
    for (int c = 0; c < 6; ++c) s_red[(x.warp * 32 + x.lane) * 6 + c] = static_cast<long long>(iacc[c]);
    __syncthreads();
    if (threadIdx.x < G * 6) {
        const int ll = threadIdx.x / 6, c = threadIdx.x % 6;
        long long v = 0;
        for (int wi = 0; wi < W; ++wi)
            for (int sb = 0; sb < SPW; ++sb) v += s_red[(wi * 32 + sb * G + ll) * 6 + c];
        const int slot = 2 * (blockIdx.z * G + ll) + c / 3;
        atomicAdd(reinterpret_cast<unsigned long long *>(x.fx) + (static_cast<size_t>(x.s) * a.R + slot) * 3 + c % 3,
                  static_cast<unsigned long long>(v));
    }
}

// ---- the kernel: one colour class (or the measure pass) per launch, so each mode gets its own register allocation
// (64 registers, no spills) and the hardware does the grid-wide ordering between colour classes.  grid (x = CTAs per
// sample and column block, y = samples of the group, z = blocks of 64 slots).
// The launches are captured in a CUDA graph with PROGRAMMATIC DEPENDENT LAUNCH edges:
// a kernel lets its successor start early (griddepcontrol.launch_dependents); the successor's CTAs become resident
// as soon as CTAs of this kernel retire, stage their graph data (sweep_prep: never theta), and only then wait for
// this kernel to complete and flush (griddepcontrol.wait).  Ramp-up thus overlaps the predecessor's tail.
// MODE 0 / 1: Metropolis / over-relaxation on colour a.t.colour; MODE 2: measure (a.t.accumulate bit 0), the last CTA
// of the sample converts the fixed-point sums; MODE 3: over-relaxation that also adds the class's share of E, Mx, My
// to the fixed-point sums (the measurement costs no extra gather), converted by the launch of the sweep's last colour.
// MODE 4 / 5 (interleaved order, xy_set_order): Metropolis and then over-relaxation of every site of the class from one
// gather, without / with the measurement by-product.

template <int G, int CB, int MODE, int W>
__global__ void __launch_bounds__(W * 32, (W == 24 || W == 28) ? 1 : kSmPerWarpSlots / W) k_phase(const SweepArgs a) {
    extern __shared__ __align__(16) unsigned char s_raw[];
    SweepWarp *s_w = reinterpret_cast<SweepWarp *>(s_raw);
    __shared__ int s_last;

    SweepCtx x;
    x.s = a.t.s0 + blockIdx.y;
    x.lane = threadIdx.x & 31;
    x.warp = threadIdx.x >> 5;
    x.sub = x.lane / G;
    x.q = blockIdx.z * G + x.lane % G;
    const uint32_t R2 = CB ? static_cast<uint32_t>(G) : static_cast<uint32_t>(a.t.R >> 1);
    x.lb = reinterpret_cast<float2 *>(a.t.theta) + static_cast<size_t>(x.s) * a.t.N * R2 + x.q;
    asm volatile("" : "+l"(x.lb));
    x.rec = a.t.rec + static_cast<size_t>(x.s) * a.t.N;
    x.sidx = s_w[x.warp].idx;
    x.ring_l = &s_w[x.warp].ring[0][0][x.lane];
    x.ring_s = static_cast<uint32_t>(__cvta_generic_to_shared(x.ring_l));
    x.fx = a.t.fx;

    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const PhasePrep P = sweep_prep<G, CB>(a, x, MODE == kModeMeasure ? kModeMeasure : kModeOverrelax, a.t.colour,
                                          gridDim.x * W, blockIdx.x * W + x.warp, true);
    __syncwarp();
    asm volatile("griddepcontrol.wait;" ::: "memory");      // the predecessor's theta / beta_slot / fx are final

    constexpr bool kTally = MODE == kModeMeasure || MODE == kModeOrMeasure || MODE == kModeMetOrMeasure;
    const uint32_t sweep = a.t.use_counter ? a.t.counters[0] + static_cast<uint32_t>(a.t.sweep_offset) : a.t.sweep_fixed;
    {
        int iacc[6] = {0, 0, 0, 0, 0, 0};
        sweep_phase<G, CB, MODE>(a.t, x, P, sweep, iacc);
        if constexpr (kTally) sweep_reduce_to_fx<G, W>(a.t, x, iacc, s_w);
    }

    if constexpr (kTally) {
        // the sums are complete after the measure launch, or after the fused launch of the sweep's last colour
        // (a.t.accumulate bit 1); its last CTA converts them
        if (MODE == kModeMeasure || (a.t.accumulate & 2)) {
            __threadfence();
            __syncthreads();
            if (threadIdx.x == 0) {
                const unsigned int total = gridDim.x * gridDim.z;
                s_last = (atomicAdd(a.t.ticket + x.s, 1u) == total - 1u) ? 1 : 0;
            }
            __syncthreads();
            if (s_last) {
                __threadfence();
                sweep_finalize(a.t, x.fx, x.s, (a.t.accumulate & 1) != 0);
                if (threadIdx.x == 0) a.t.ticket[x.s] = 0u;
            }
        }
    }
}

}  // namespace xy
