// xy_w32.cuh -- the R % 64 == 0 flavour of the colour-class kernels (config 4: R = 64): one warp = one site,
// one lane = two adjacent slots (float2), software-pipelined across sites through shared memory.
//
// Why a second kernel (profiles/r1a_full.md, r1b_full.md): the path is bound by instruction
// issue and latency, not by bytes.  The tile kernel issues a site's gathers and then waits for them
// (long_scoreboard 7 of 11 stall cycles per issue, issue slots 50 % busy); holding the in-flight gathers of
// the next site in registers costs 120 registers and leaves 16 warps per SM.  Same-colour sites share no
// bond, so the gathers of site t+1 never read what site t stores: they are issued BEFORE site
// t is computed, as cp.async (LDGSTS) copies of the lane's own 8 bytes into a per-warp ring in shared
// memory.  In-flight data then costs no registers (<= 64 per thread, 32 warps per SM), each lane reads back
// only what it copied itself (no cross-lane synchronisation, cp.async.wait_group only), and the Philox /
// sin / exp work of site t covers the latency of site t+1.
// Per neighbour a lane issues: one broadcast LDS (pre-scaled id), one IMAD.WIDE address, one LDGSTS (a
// 256-byte request per warp), one LDS.64, and packed fp32x2 arithmetic (add/mul.rn.f32x2 -> FADD2/FMUL2 on
// sm_100a) for its two slots.
//
// A warp owns a contiguous, equal share of the colour class and walks it in chunks of <= 32 sites: one
// coalesced load of the chunk's rec[], the chunk's neighbour ids (one contiguous CSR run) staged in the
// warp's slice of shared memory.  Neighbours beyond kDB per site use a short non-pipelined tail loop; a
// single site whose degree exceeds the staging capacity is walked in blocks.
#pragma once
#include "xy_kernels.cuh"

namespace xy {

constexpr int kDB = 8;            // pipelined gathers per site
constexpr int kDepth = 2;         // ring slots per warp (sites in flight)
constexpr int kStageCap = 256;    // staged neighbour ids per warp and chunk (ints)
#ifndef XY_W32_MIN_BLOCKS
#define XY_W32_MIN_BLOCKS 4
#endif
constexpr int kW32MinBlocks = XY_W32_MIN_BLOCKS;  // resident CTAs per SM the register / shared budget is sized for

// per warp: ring[kDepth][kDB + 1][32] float2 (row kDB = the site's own angle) + staged ids
struct __align__(16) W32Warp {
    float2 ring[kDepth][kDB + 1][32];
    uint32_t idx[kStageCap];
};
static_assert(sizeof(W32Warp) * kWarps <= 48 * 1024 - 64, "static shared memory limit");
static_assert(sizeof(W32Warp) * kWarps >= sizeof(double) * kWarps * 32 * 6, "measure reduction reuses the ring");

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

// ---- cp.async (LDGSTS): 8 bytes per lane, global -> shared, no register staging ---------------------------
__device__ __forceinline__ void cp_async8(uint32_t smem_addr, const void *gptr) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_addr), "l"(gptr));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- per-lane state of one site (two slots) ----------------------------------------------------------
template <int MODE> struct PairAcc;
template <> struct PairAcc<kModeMetropolis> {
    float2 mid, s = make_float2(0.f, 0.f);
    __device__ __forceinline__ void add(const float2 t) {
        const float2 d = sub2(mid, t);
        s = add2(s, make_float2(__sinf(d.x), __sinf(d.y)));
    }
};
template <> struct PairAcc<kModeOverrelax> {
    float2 hx = make_float2(0.f, 0.f), hy = make_float2(0.f, 0.f);   // hx = (h_x of slot .x, h_x of slot .y)
    __device__ __forceinline__ void add(const float2 t) {
        float sx, cx, sy, cy;
        __sincosf(t.x, &sx, &cx);
        __sincosf(t.y, &sy, &cy);
        hx = add2(hx, make_float2(cx, cy));
        hy = add2(hy, make_float2(sx, sy));
    }
};
template <> struct PairAcc<kModeMeasure> {
    float2 own, e = make_float2(0.f, 0.f);
    __device__ __forceinline__ void add(const float2 t) {
        const float2 d = sub2(own, t);
        e = add2(e, make_float2(__cosf(d.x), __cosf(d.y)));
    }
};

struct W32Site { int i, deg, pos; };   // warp-uniform: site id, neighbours to visit, first staged id

// direct gather of the neighbour with pre-scaled id `sid` (float2 units): one IMAD.WIDE.U32 + one LDG.64
__device__ __forceinline__ float2 w32_ld(const float2 *lb, uint32_t sid) {
    return __ldcg(lb + static_cast<unsigned long long>(sid));
}

template <int D>
__device__ __forceinline__ void w32_issue_n(uint32_t row0, const float2 *lb, const uint32_t *sidx, int pos) {
    uint32_t sid[D];
#pragma unroll
    for (int u = 0; u < D; ++u) sid[u] = sidx[pos + u];      // all id loads first: LDS -> LDGSTS hazards are paid once
#pragma unroll
    for (int u = 0; u < D; ++u) cp_async8(row0 + u * 256u, lb + static_cast<unsigned long long>(sid[u]));
}

// issue min(deg, kDB) async gathers back to back (deg is warp-uniform: exact count, nothing predicated off);
// row0 = shared address of this lane's 8 bytes in row 0 of the ring slot
__device__ __forceinline__ void w32_issue(uint32_t row0, const float2 *lb, const uint32_t *sidx, int pos, int deg) {
    switch (deg < kDB ? deg : kDB) {
        case 8: w32_issue_n<8>(row0, lb, sidx, pos); break;
        case 7: w32_issue_n<7>(row0, lb, sidx, pos); break;
        case 6: w32_issue_n<6>(row0, lb, sidx, pos); break;
        case 5: w32_issue_n<5>(row0, lb, sidx, pos); break;
        case 4: w32_issue_n<4>(row0, lb, sidx, pos); break;
        case 3: w32_issue_n<3>(row0, lb, sidx, pos); break;
        case 2: w32_issue_n<2>(row0, lb, sidx, pos); break;
        case 1: w32_issue_n<1>(row0, lb, sidx, pos); break;
        default: break;
    }
}

template <int D, typename ACC>
__device__ __forceinline__ void w32_consume_n(ACC &acc, const float2 *row0) {
    float2 v[D];
#pragma unroll
    for (int u = 0; u < D; ++u) v[u] = row0[u * 32];
#pragma unroll
    for (int u = 0; u < D; ++u) acc.add(v[u]);
}

// row0 = pointer to this lane's float2 in row 0 of the ring slot
template <typename ACC>
__device__ __forceinline__ void w32_consume(ACC &acc, const float2 *row0, const float2 *lb, const uint32_t *sidx,
                                            int pos, int deg) {
    switch (deg < kDB ? deg : kDB) {
        case 8: w32_consume_n<8>(acc, row0); break;
        case 7: w32_consume_n<7>(acc, row0); break;
        case 6: w32_consume_n<6>(acc, row0); break;
        case 5: w32_consume_n<5>(acc, row0); break;
        case 4: w32_consume_n<4>(acc, row0); break;
        case 3: w32_consume_n<3>(acc, row0); break;
        case 2: w32_consume_n<2>(acc, row0); break;
        case 1: w32_consume_n<1>(acc, row0); break;
        default: break;
    }
    for (int k = kDB; k < deg; k += 4) {   // rare tail (more than kDB neighbours), not pipelined
        float2 t[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (k + u < deg) t[u] = w32_ld(lb, sidx[pos + k + u]);
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (k + u < deg) acc.add(t[u]);
    }
}

// ---- the kernel ----------------------------------------------------------------------------------------
// grid (x = CTAs per sample and column block, y = samples of the group, z = blocks of 64 slots).
// CB = 1: R == 64 (stride known at compile time).  MODE as in k_tile.
template <int CB, int MODE>
__global__ void __launch_bounds__(kBlock, kW32MinBlocks) k_w32(const TileArgs a) {
    __shared__ W32Warp s_w[kWarps];
    __shared__ int s_last;

    const int s = a.s0 + blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t R2 = CB ? 32u : static_cast<uint32_t>(a.R >> 1);
    const int q = blockIdx.z * 32 + lane;          // slot pair handled by this lane

    int cbeg = 0, cend = a.N;
    if constexpr (MODE != kModeMeasure) {
        cbeg = a.class_ptr[s * a.q_stride + a.colour];
        cend = a.class_ptr[s * a.q_stride + a.colour + 1];
    }
    // contiguous equal shares of the class over the warps of this (sample, column block)
    const int nw = gridDim.x * kWarps, gw = blockIdx.x * kWarps + warp;
    const int per = (cend - cbeg + nw - 1) / nw;
    const int w0 = min(cend, cbeg + gw * per), w1 = min(cend, w0 + per);

    float2 *lb = reinterpret_cast<float2 *>(a.theta) + static_cast<size_t>(s) * a.N * R2 + q;
    asm volatile("" : "+l"(lb));   // keep the lane's base as one materialised pointer: gather address = one IMAD.WIDE.U32
    const int2 *__restrict__ rec = a.rec + static_cast<size_t>(s) * a.N;
    uint32_t *sidx = s_w[warp].idx;
    const float2 *ring_l = &s_w[warp].ring[0][0][lane];                       // this lane's column of the ring
    const uint32_t ring_s = static_cast<uint32_t>(__cvta_generic_to_shared(ring_l));
    constexpr uint32_t kSlotBytes = (kDB + 1) * 32 * sizeof(float2);
    constexpr int kSlotElems = (kDB + 1) * 32;

    float2 nbeta = make_float2(0.f, 0.f), w = make_float2(0.f, 0.f);
    uint32_t sweep = 0, c2 = 0;
    if constexpr (MODE == kModeMetropolis) {
        const float2 b = reinterpret_cast<const float2 *>(a.beta_slot)[static_cast<size_t>(s) * R2 + q];
        nbeta = make_float2(-b.x, -b.y);
        w = reinterpret_cast<const float2 *>(a.w_slot)[static_cast<size_t>(s) * R2 + q];
        sweep = a.use_counter ? a.counters[0] + static_cast<uint32_t>(a.sweep_offset) : a.sweep_fixed;
        c2 = ((a.sample_base + static_cast<uint32_t>(s)) << 16) | static_cast<uint32_t>(q);
    }
    double dacc[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};   // measure: E, Mx, My of the .x slot, then of the .y slot

    // Metropolis proposal of site i (both slots of the lane): th' = th + w (u1 - 1/2), half = (th' - th)/2
    auto begin = [&](int i, const float2 own, PairAcc<MODE> &acc, float2 &thp, float2 &half, float2 &u2) {
        if constexpr (MODE == kModeMetropolis) {
            uint32_t x[4];
            philox4x32_10(static_cast<uint32_t>(i), sweep, c2, kDomMetropolis, a.keys, x);
            // u = (k + 1/2) 2^-23 with k = x >> 9 (R11), every step exact:
            //   u1 - 1/2 = ((1 + k 2^-23) - 3/2) + 2^-24,   u2 = (1 + k 2^-23) - (1 - 2^-24)
            const float2 u1mh = add2(add2(make_float2(mant12(x[0]), mant12(x[2])), make_float2(-1.5f, -1.5f)),
                                     make_float2(5.9604644775390625e-08f, 5.9604644775390625e-08f));
            u2 = add2(make_float2(mant12(x[1]), mant12(x[3])), make_float2(-0.99999994f, -0.99999994f));
            thp = add2(own, mul2(w, u1mh));                      // R5: fp32 mul, fp32 add
            half = mul2(sub2(thp, own), make_float2(0.5f, 0.5f));
            acc.mid = add2(own, half);
        } else if constexpr (MODE == kModeMeasure) {
            acc.own = own;
        }
    };
    auto finish = [&](int i, const float2 own, const PairAcc<MODE> &acc, const float2 thp, const float2 half,
                      const float2 u2, float2 &fe, float2 &fmx, float2 &fmy) {
        if constexpr (MODE == kModeMetropolis) {
            // dE = 2 sin((th'-th)/2) sum_j sin((th'+th)/2 - th_j)
            const float2 sh = make_float2(__sinf(half.x), __sinf(half.y));
            const float2 arg = mul2(nbeta, mul2(add2(sh, sh), acc.s));
            float2 out;
            out.x = metropolis_select(own.x, thp.x, u2.x, __expf(arg.x));
            out.y = metropolis_select(own.y, thp.y, u2.y, __expf(arg.y));
            lb[static_cast<unsigned long long>(static_cast<uint32_t>(i) * R2)] = out;
        } else if constexpr (MODE == kModeOverrelax) {
            float2 out;
            out.x = overrelax_finish(own.x, acc.hx.x, acc.hy.x);
            out.y = overrelax_finish(own.y, acc.hx.y, acc.hy.y);
            lb[static_cast<unsigned long long>(static_cast<uint32_t>(i) * R2)] = out;
        } else {
            float sx, cx, sy, cy;
            __sincosf(own.x, &sx, &cx);
            __sincosf(own.y, &sy, &cy);
            fe = add2(fe, acc.e);
            fmx = add2(fmx, make_float2(cx, cy));
            fmy = add2(fmy, make_float2(sx, sy));
        }
    };

    for (int i0 = w0; i0 < w1;) {
        // ---- chunk: the longest prefix of <= 32 sites whose neighbour ids fit the staging slice ----
        const int nsite = min(32, w1 - i0);
        int2 rc = make_int2(0, 0);
        if (lane < nsite) rc = rec[i0 + lane];
        const int start0 = __shfl_sync(kFull, rc.x, 0);
        const int endl = rc.x + (rc.y & 0xffff) - start0;
        const unsigned fits = __ballot_sync(kFull, lane < nsite && endl <= kStageCap);
        const int msite = fits == kFull ? 32 : __ffs(~fits) - 1;      // leading sites that fit
        float2 fe = make_float2(0.f, 0.f), fmx = make_float2(0.f, 0.f), fmy = make_float2(0.f, 0.f);

        if (msite == 0) {
            // a single site with more neighbours than the staging slice: walk its ids in blocks
            const int ry = __shfl_sync(kFull, rc.y, 0);
            int deg = ry & 0xffff, pos = 0;
            if constexpr (MODE == kModeMeasure) { pos = ry >> 16; deg -= pos; }
            const int32_t *gidx = a.col_idx + start0 + pos;
            const float2 own = lb[static_cast<unsigned long long>(static_cast<uint32_t>(i0) * R2)];
            float2 thp = make_float2(0.f, 0.f), half = thp, u2 = thp;
            PairAcc<MODE> acc;
            begin(i0, own, acc, thp, half, u2);
            for (int k0 = 0; k0 < deg; k0 += kStageCap) {
                const int nb = min(kStageCap, deg - k0);
                __syncwarp();
                for (int p = lane; p < nb; p += 32) sidx[p] = static_cast<uint32_t>(gidx[k0 + p]) * R2;
                __syncwarp();
                for (int k = 0; k < nb; k += 4) {
                    float2 t[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        if (k + u < nb) t[u] = w32_ld(lb, sidx[k + u]);
#pragma unroll
                    for (int u = 0; u < 4; ++u)
                        if (k + u < nb) acc.add(t[u]);
                }
            }
            finish(i0, own, acc, thp, half, u2, fe, fmx, fmy);
            __syncwarp();
            i0 += 1;
        } else {
            const int n_run = __shfl_sync(kFull, endl, msite - 1);
            const int32_t *gidx = a.col_idx + start0;
            for (int p0 = 0; p0 < n_run; p0 += 128) {       // stage (pre-scaled by the site stride): 4 loads in flight
                int32_t g[4];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (p0 + u * 32 + lane < n_run) g[u] = gidx[p0 + u * 32 + lane];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (p0 + u * 32 + lane < n_run) sidx[p0 + u * 32 + lane] = static_cast<uint32_t>(g[u]) * R2;
            }
            __syncwarp();

            auto site_of = [&](int t) {
                const int ry = __shfl_sync(kFull, rc.y, t), rx = __shfl_sync(kFull, rc.x, t);
                W32Site st{i0 + t, ry & 0xffff, rx - start0};
                if constexpr (MODE == kModeMeasure) {     // bonds counted once: neighbours j > i are the tail of the list
                    st.pos += ry >> 16;
                    st.deg -= ry >> 16;
                }
                return st;
            };
            // async copies of site st (own angle -> row kDB, first kDB neighbours -> rows 0..) into ring slot `slot`
            auto issue = [&](const W32Site st, int slot) {
                const uint32_t row0 = ring_s + static_cast<uint32_t>(slot) * kSlotBytes;
                cp_async8(row0 + kDB * 256u, lb + static_cast<unsigned long long>(static_cast<uint32_t>(st.i) * R2));
                w32_issue(row0, lb, sidx, st.pos, st.deg);
                cp_async_commit();
            };

            // software pipeline over the chunk: the copies of site t+1 fly while site t is computed
            W32Site cur = site_of(0);
            issue(cur, 0);
            for (int t = 0; t < msite; ++t) {
                W32Site nxt = cur;
                if (t + 1 < msite) {
                    nxt = site_of(t + 1);
                    issue(nxt, (t + 1) & 1);
                    cp_async_wait<1>();
                } else {
                    cp_async_wait<0>();
                }
                const float2 *row0 = ring_l + (t & 1) * kSlotElems;
                const float2 own = row0[kDB * 32];
                float2 thp = make_float2(0.f, 0.f), half = thp, u2 = thp;
                PairAcc<MODE> acc;
                begin(cur.i, own, acc, thp, half, u2);
                w32_consume(acc, row0, lb, sidx, cur.pos, cur.deg);
                finish(cur.i, own, acc, thp, half, u2, fe, fmx, fmy);
                cur = nxt;
            }
            __syncwarp();
            i0 += msite;
        }
        if constexpr (MODE == kModeMeasure) {
            dacc[0] -= static_cast<double>(fe.x); dacc[1] += static_cast<double>(fmx.x); dacc[2] += static_cast<double>(fmy.x);
            dacc[3] -= static_cast<double>(fe.y); dacc[4] += static_cast<double>(fmx.y); dacc[5] += static_cast<double>(fmy.y);
        }
    }

    if constexpr (MODE == kModeMeasure) {
        // CTA reduction in a fixed order (the ring is free now), then exact order-independent fixed-point accumulation
        __syncthreads();
        double *s_red = reinterpret_cast<double *>(&s_w[0]);
#pragma unroll
        for (int c = 0; c < 6; ++c) s_red[(warp * 32 + lane) * 6 + c] = dacc[c];
        __syncthreads();
        if (threadIdx.x < 32 * 6) {
            const int ll = threadIdx.x / 6, c = threadIdx.x % 6;
            double v = 0.0;
            for (int wi = 0; wi < kWarps; ++wi) v += s_red[(wi * 32 + ll) * 6 + c];
            const int slot = 2 * (blockIdx.z * 32 + ll) + c / 3;
            atomicAdd(reinterpret_cast<unsigned long long *>(a.fx) + (static_cast<size_t>(s) * a.R + slot) * 3 + c % 3,
                      static_cast<unsigned long long>(__double2ll_rn(v * kFix)));
        }
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) {
            const unsigned int total = gridDim.x * gridDim.z;
            s_last = (atomicAdd(a.ticket + s, 1u) == total - 1u) ? 1 : 0;
        }
        __syncthreads();
        if (s_last) {
            __threadfence();
            measure_finalize(a, s);
        }
    }
}

}  // namespace xy
