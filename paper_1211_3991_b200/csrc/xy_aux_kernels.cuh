// xy_aux_kernels.cuh -- the kernels outside the colour-class hot loop (included by xy_b200.cu only): the any-R path (one
// warp per site, lanes stride over the slots; one launch per colour class) that serves replica counts without a float2
// flavour (odd R, R = 6, 10, ...), the structure factor at k_min, the random-walk return histogram, the angle
// initialisation, the stand-alone swap round and the counter tick.
//
// PAPER.md:444,:454 (coloured single-spin Metropolis), :460 (over-relaxation, ref 66), :167-181 (E, m), :183-190 (chi(k)),
// :436-440 (random walks), :460-472 (parallel tempering); readings R5-R11, R18, R19 in DESIGN.md.
#pragma once
#include <type_traits>

#include "xy_kernels.cuh"

namespace xy {

// last CTA of a sample: fixed-point sums -> E, M per slot; optional accumulation under the slot's temperature
// (Eq. 13-16); leaves fx and the ticket zeroed for the next launch
__device__ __forceinline__ void measure_finalize(const TileArgs &a, int s) {
    for (int r = threadIdx.x; r < a.R; r += blockDim.x) {
        long long *f = a.fx + (static_cast<size_t>(s) * a.R + r) * 3;
        const double e = static_cast<double>(__ldcg(f)) * kInvFix;
        const double mx = static_cast<double>(__ldcg(f + 1)) * kInvFix;
        const double my = static_cast<double>(__ldcg(f + 2)) * kInvFix;
        f[0] = 0; f[1] = 0; f[2] = 0;
        const size_t sr = static_cast<size_t>(s) * a.R + r;
        a.E_slot[sr] = e;
        a.M_slot[2 * sr] = mx;
        a.M_slot[2 * sr + 1] = my;
        if (a.accumulate) {
            double *o = a.acc + (static_cast<size_t>(s) * a.R + a.temp_of_slot[sr]) * 8;
            const double ux = mx / a.N, uy = my / a.N, m2 = ux * ux + uy * uy;
            o[0] += 1.0; o[1] += e; o[2] += e * e; o[3] += sqrt(m2); o[4] += m2; o[5] += m2 * m2;
            o[6] += ux; o[7] += uy;
        }
    }
    if (threadIdx.x == 0) a.ticket[s] = 0u;
}

// ---- generic path: any R >= 1 (odd R, R = 6, ...): one warp per site, lanes stride over the slots ----
template <int MODE>
__global__ void __launch_bounds__(kBlock) k_update_class_generic(const TileArgs a) {
    const int s = a.s0 + blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int cbeg = a.class_ptr[s * a.q_stride + a.colour];
    const int cend = a.class_ptr[s * a.q_stride + a.colour + 1];
    const int n_sites = cend - cbeg;
    const int g0 = (blockIdx.x * kWarps + warp) * a.tiles_per_warp;
    if (g0 >= n_sites) return;
    const int g1 = min(g0 + a.tiles_per_warp, n_sites);
    float *__restrict__ th = a.theta + static_cast<size_t>(s) * a.N * a.R;
    const int2 *__restrict__ rec = a.rec + static_cast<size_t>(s) * a.N;
    const uint32_t sweep = a.use_counter ? a.counters[0] + static_cast<uint32_t>(a.sweep_offset) : a.sweep_fixed;

    for (int g = g0; g < g1; ++g) {
        const int i = cbeg + g;
        const int2 rc = rec[i];
        const int deg = rc.y & 0xffff;
        for (int r = lane; r < a.R; r += 32) {
            const float own = th[static_cast<size_t>(i) * a.R + r];
            float thp = 0.f, half = 0.f, mid = 0.f, u2 = 0.f, acc0 = 0.f, acc1 = 0.f;
            if (MODE == kModeMetropolis) {
                uint32_t x[4];
                philox4x32_10(static_cast<uint32_t>(i), sweep,
                              ((a.sample_base + static_cast<uint32_t>(s)) << 16) | static_cast<uint32_t>(r >> 1),
                              kDomMetropolis, a.keys, x);
                const float u1 = (r & 1) ? u01(x[2]) : u01(x[0]);
                u2 = (r & 1) ? u01(x[3]) : u01(x[1]);
                const float w = a.w_slot[static_cast<size_t>(s) * a.R + r];
                thp = __fadd_rn(own, __fmul_rn(w, u1 - 0.5f));
                half = 0.5f * (thp - own);
                mid = own + half;
            }
            for (int e = 0; e < deg; ++e) {
                const float t = th[static_cast<size_t>(a.col_idx[rc.x + e]) * a.R + r];
                if (MODE == kModeMetropolis) {
                    acc0 += __sinf(mid - t);
                } else {
                    float sn, cs;
                    __sincosf(t, &sn, &cs);
                    acc0 += cs; acc1 += sn;
                }
            }
            float out;
            if (MODE == kModeMetropolis)
                // dE = -sum_j[cos(th' - th_j) - cos(th - th_j)] = 2 sin((th'-th)/2) sum_j sin((th'+th)/2 - th_j)
                out = metropolis_select(own, thp, u2,
                                        __expf(-a.beta_slot[static_cast<size_t>(s) * a.R + r] * (2.0f * __sinf(half) * acc0)));
            else
                out = overrelax_finish(own, acc0, acc1);
            th[static_cast<size_t>(i) * a.R + r] = out;
        }
    }
}

// generic measure: grid (n_chunks, samples); thread = slot (strided), sequential over the CTA's sites
__global__ void __launch_bounds__(kBlock) k_measure_generic(const TileArgs a, int chunk_sites) {
    __shared__ int s_last;
    const int s = a.s0 + blockIdx.y;
    const int ibeg = blockIdx.x * chunk_sites;
    const int iend = min(ibeg + chunk_sites, a.N);
    const float *__restrict__ th = a.theta + static_cast<size_t>(s) * a.N * a.R;
    const int2 *__restrict__ rec = a.rec + static_cast<size_t>(s) * a.N;
    for (int r = threadIdx.x; r < a.R; r += kBlock) {
        double e = 0.0, mx = 0.0, my = 0.0;
        for (int i = ibeg; i < iend; ++i) {
            const int2 rc = rec[i];
            const int deg = rc.y & 0xffff, nlow = static_cast<int>(static_cast<uint32_t>(rc.y) >> 16);
            const float own = th[static_cast<size_t>(i) * a.R + r];
            float sn, cs, es = 0.f;
            __sincosf(own, &sn, &cs);
            for (int k = nlow; k < deg; ++k)
                es += __cosf(own - th[static_cast<size_t>(a.col_idx[rc.x + k]) * a.R + r]);
            e -= static_cast<double>(es); mx += static_cast<double>(cs); my += static_cast<double>(sn);
        }
        unsigned long long *f = reinterpret_cast<unsigned long long *>(a.fx) + (static_cast<size_t>(s) * a.R + r) * 3;
        atomicAdd(f, static_cast<unsigned long long>(__double2ll_rn(e * kFix)));
        atomicAdd(f + 1, static_cast<unsigned long long>(__double2ll_rn(mx * kFix)));
        atomicAdd(f + 2, static_cast<unsigned long long>(__double2ll_rn(my * kFix)));
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(a.ticket + s, 1u) == gridDim.x - 1u) ? 1 : 0;
    __syncthreads();
    if (s_last) {
        __threadfence();
        measure_finalize(a, s);
    }
}

// ---- structure factor at the smallest momenta (Eq. 17-18) ---------------
// G1 = |sum_i S_i exp(i 2 pi x_i / Lx)|^2 / N, G2 likewise with y_i / Ly, per (sample, slot): the single-configuration
// estimators of chi(k_min).  One streaming pass over theta (4 bytes per spin and slot, no gathers): a warp walks a
// contiguous range of sites, lane = slot (blocks of 32 slots), eight sums per slot (Re/Im x two spin components x
// two momenta) as exact fixed-point integers (scale 2^22, see quant of the measure kernel), so the result does not
// depend on the grid.  The last CTA of a sample converts the sums and files G1, G2 under the slot's temperature.
struct FourierArgs {
    const float *theta;             // [S][N][R]
    const uint32_t *coords;         // [S][N] x | y << 16
    const float2 *tab1, *tab2;      // [Lx], [Ly]: (cos, sin)(2 pi n / L)
    long long *fk;                  // [S][R][8] fixed-point sums, zero between launches
    unsigned int *ticket;           // [S]
    const int32_t *temp_of_slot;    // [S][R]
    double *G_slot;                 // [S][R][2]
    double *acc_k;                  // [S][R][3]: n, sum G1, sum G2 by temperature
    int N, R, s0, sites_per_warp;
};

__device__ __forceinline__ int quant_unit(float x) { return __float_as_int(__fadd_rn(x, 3.0f)) - 0x40400000; }   // rn(x 2^22), |x| <= 1

__global__ void __launch_bounds__(kBlock) k_fourier(const FourierArgs a) {
    __shared__ int s_last;
    const int s = a.s0 + blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int i0 = (blockIdx.x * kWarps + warp) * a.sites_per_warp;
    const int i1 = min(a.N, i0 + a.sites_per_warp);
    const float *th = a.theta + static_cast<size_t>(s) * a.N * a.R;
    const uint32_t *co = a.coords + static_cast<size_t>(s) * a.N;
    for (int r = lane; r < a.R && i0 < i1; r += 32) {
        long long acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        int part[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        int n_part = 0;
        for (int i = i0; i < i1; ++i) {
            const uint32_t xy = __ldg(co + i);
            const float2 p1 = __ldg(a.tab1 + (xy & 0xffffu)), p2 = __ldg(a.tab2 + (xy >> 16));
            float sn, cs;
            __sincosf(th[static_cast<size_t>(i) * a.R + r], &sn, &cs);
            part[0] += quant_unit(__fmul_rn(cs, p1.x)); part[1] += quant_unit(__fmul_rn(cs, p1.y));
            part[2] += quant_unit(__fmul_rn(sn, p1.x)); part[3] += quant_unit(__fmul_rn(sn, p1.y));
            part[4] += quant_unit(__fmul_rn(cs, p2.x)); part[5] += quant_unit(__fmul_rn(cs, p2.y));
            part[6] += quant_unit(__fmul_rn(sn, p2.x)); part[7] += quant_unit(__fmul_rn(sn, p2.y));
            if (++n_part == 256) {      // 256 * 2^22 < 2^31
#pragma unroll
                for (int c = 0; c < 8; ++c) { acc[c] += part[c]; part[c] = 0; }
                n_part = 0;
            }
        }
        unsigned long long *f = reinterpret_cast<unsigned long long *>(a.fk) + (static_cast<size_t>(s) * a.R + r) * 8;
#pragma unroll
        for (int c = 0; c < 8; ++c) atomicAdd(f + c, static_cast<unsigned long long>(acc[c] + part[c]));
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(a.ticket + s, 1u) == gridDim.x - 1u) ? 1 : 0;
    __syncthreads();
    if (s_last) {
        __threadfence();
        const double inv = 1.0 / 4194304.0;
        for (int r = threadIdx.x; r < a.R; r += blockDim.x) {
            long long *f = a.fk + (static_cast<size_t>(s) * a.R + r) * 8;
            double v[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) { v[c] = static_cast<double>(__ldcg(f + c)) * inv; f[c] = 0; }
            const double g1 = (v[0] * v[0] + v[1] * v[1] + v[2] * v[2] + v[3] * v[3]) / a.N;
            const double g2 = (v[4] * v[4] + v[5] * v[5] + v[6] * v[6] + v[7] * v[7]) / a.N;
            const size_t sr = static_cast<size_t>(s) * a.R + r;
            a.G_slot[2 * sr] = g1;
            a.G_slot[2 * sr + 1] = g2;
            double *o = a.acc_k + (static_cast<size_t>(s) * a.R + a.temp_of_slot[sr]) * 3;
            o[0] += 1.0; o[1] += g1; o[2] += g2;
        }
        if (threadIdx.x == 0) a.ticket[s] = 0u;
    }
}

// packed fp32x2 helpers of k_fourier2 (one FFMA2 serves the lane's two slots)
__device__ __forceinline__ void fma2(unsigned long long &acc, unsigned long long a, unsigned long long b) {
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(a), "l"(b));
}
__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ float2 unpack2(unsigned long long v) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}

// float2 flavour of k_fourier for R = 2G (G a power of two <= 32) or R a multiple of 64 (G = 32, blockIdx.z = block
// of 64 slots): a lane owns two adjacent slots, G lanes cover a site, a warp reads 32/G sites per row (one fully used
// 256-byte request at R >= 64).  The pass is a pure stream and the kernel is bound by ISSUE SLOTS, not by bytes in flight
// (ncu, profiles/r2b_fourier.md: 64 instructions per row at 69 % issue utilisation), so the row is stripped to the bone:
//   * a ring of kFourierRing rows per warp filled by cp.async copies of the lane's own 8 bytes (no registers held by
//     loads in flight, 128 KB per SM on their way), ring slots at compile-time offsets, the source offset a running 32-bit
//     count, no bounds test on full blocks (the last block of a warp's range runs the predicated variant);
//   * the site's phase factors (cos, sin)(2 pi x / Lx), (cos, sin)(2 pi y / Ly): lane l loads the coordinates of site
//     32 b + l two blocks ahead and its table entries one block ahead (no exposed latency; the tables need not survive in
//     L1, which the stream flushes) and posts the four values in shared memory; a row reads its site's with one LDS.128;
//   * 4 MUFU + 8 packed FFMA2 (fp32x2, the factor as the scalar operand) for the lane's two slots.
// Same fixed-point sums, same finalisation as k_fourier.
constexpr int kFourierRing = 16;
constexpr int kFourierStageRows = 4;                                   // BULK: rows per bulk copy (1 KB) and mbarrier
constexpr int kFourierStages = kFourierRing / kFourierStageRows;
struct __align__(16) FourierWarp {
    float2 ring[kFourierRing][32];
    float4 fac[32];
    unsigned long long bar[kFourierStages];      // BULK: one mbarrier per stage of the ring
};

// ---- bulk asynchronous copies (cp.async.bulk: the TMA engine moves a contiguous run global -> shared without passing
// L1TEX and signals an mbarrier with the bytes it delivered) ----
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "FOURIER_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra FOURIER_DONE;\n"
        "bra FOURIER_WAIT;\n"
        "FOURIER_DONE:\n"
        "}" ::"r"(bar), "r"(parity) : "memory");
}

constexpr size_t kFourierRed = sizeof(long long) * kWarps * 32 * 16;
constexpr size_t kFourierSmem = sizeof(FourierWarp) * kWarps > kFourierRed ? sizeof(FourierWarp) * kWarps : kFourierRed;

template <int G, bool BULK>
__global__ void __launch_bounds__(kBlock, 4) k_fourier2(const FourierArgs a) {
    constexpr int SPW = 32 / G;
    constexpr int NS = kFourierRing;
    constexpr int RPB = 32 / SPW;         // rows per block of 32 sites
    constexpr bool kConstSlots = RPB % NS == 0;
    extern __shared__ __align__(16) unsigned char f_raw[];
    __shared__ int s_last;
    const int s = a.s0 + blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sub = lane / G, q = blockIdx.z * G + lane % G;           // slot pair of this lane
    const uint32_t R2 = static_cast<uint32_t>(a.R >> 1);
    const int i0 = (blockIdx.x * kWarps + warp) * a.sites_per_warp;
    const int i1 = min(a.N, i0 + a.sites_per_warp);
    const float2 *th = reinterpret_cast<const float2 *>(a.theta) + static_cast<size_t>(s) * a.N * R2 + q;
    const uint32_t *co = a.coords + static_cast<size_t>(s) * a.N;
    FourierWarp *fw = reinterpret_cast<FourierWarp *>(f_raw) + warp;
    const float2 *ring_l = &fw->ring[0][lane];
    const uint32_t ring_s = static_cast<uint32_t>(__cvta_generic_to_shared(ring_l));
    // eight packed fp32x2 partial sums over <= 256 rows of the lane's own range: P[c] = (sum c of the lane's even slot,
    // of its odd slot).  Fixed order (the partition is a function of N, S and R only), so a run is bit-reproducible;
    // exact fixed-point sums across flushes, warps and CTAs.
    unsigned long long P[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) P[c] = 0ull;
    // f = (c1, s1, c2, s2) = (cos, sin)(2 pi x / Lx), (cos, sin)(2 pi y / Ly) of the row's site
    auto tally = [&](const float2 t, const float4 f) {
        float sx, cx, sy, cy;
        __sincosf(t.x, &sx, &cx);
        __sincosf(t.y, &sy, &cy);
        const unsigned long long cs = pack2(cx, cy), sn = pack2(sx, sy);
        const unsigned long long c1p = pack2(f.x, f.x), s1p = pack2(f.y, f.y), c2p = pack2(f.z, f.z), s2p = pack2(f.w, f.w);
        fma2(P[0], cs, c1p); fma2(P[1], cs, s1p); fma2(P[2], sn, c1p); fma2(P[3], sn, s1p);
        fma2(P[4], cs, c2p); fma2(P[5], cs, s2p); fma2(P[6], sn, c2p); fma2(P[7], sn, s2p);
    };
    float part[16];                      // [0..7] the even slot's sums, [8..15] the odd slot's (unpacked at a flush only)
    auto unpack = [&]() {
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const float2 v = unpack2(P[c]);
            part[c] = v.x; part[8 + c] = v.y;
            P[c] = 0ull;
        }
    };
    auto flush = [&]() {      // rare (once per 256 rows and lane): no 64-bit accumulators live in the loop
        unsigned long long *f = reinterpret_cast<unsigned long long *>(a.fk) + (static_cast<size_t>(s) * a.R + 2 * q) * 8;
        unpack();
#pragma unroll
        for (int c = 0; c < 16; ++c)
            atomicAdd(f + c, static_cast<unsigned long long>(__double2ll_rn(static_cast<double>(part[c]) * 4194304.0)));
    };
    // row r of the warp = sites i0 + r SPW + sub; its copy lands in ring slot r % NS.  n_full = rows whose SPW sites all exist.
    const int n_rows = i0 < i1 ? (i1 - i0 + SPW - 1) / SPW : 0;
    const int n_full = i0 < i1 ? (i1 - i0) / SPW : 0;
    uint32_t off = static_cast<uint32_t>(i0 + sub) * R2;        // float2 offset of the next row to issue (N R / 2 < 2^31)
    int r_issue = 0;
    auto issue = [&](auto full, int slot) {     // copy of row r_issue into ring slot `slot`; one group per row, empty or not
        if constexpr (!BULK) {
            if (decltype(full)::value || (r_issue < n_rows && i0 + r_issue * SPW + sub < i1))
                cp_async8(ring_s + static_cast<uint32_t>(slot) * 256u, th + static_cast<unsigned long long>(off));
            cp_async_commit();
            off += SPW * R2;
            r_issue += 1;
        }
    };
    // BULK: the ring is filled a stage (kFourierStageRows rows, 1 KB) at a time by lane 0: one bulk copy when the rows
    // are contiguous in memory (R = 2 G: one column block), else one per row; the stage's mbarrier counts the bytes
    constexpr int RS = kFourierStageRows, NST = kFourierStages;
    const uint32_t bar_s = static_cast<uint32_t>(__cvta_generic_to_shared(&fw->bar[0]));
    const uint32_t stage_s = static_cast<uint32_t>(__cvta_generic_to_shared(&fw->ring[0][0]));
    const unsigned char *row_src = reinterpret_cast<const unsigned char *>(
        reinterpret_cast<const float2 *>(a.theta) + static_cast<size_t>(s) * a.N * R2 + blockIdx.z * G);      // + 8 R2 per site
    auto issue_stage = [&](int st) {
        if (st * RS < n_rows && lane == 0) {
            const uint32_t bar = bar_s + static_cast<uint32_t>(st % NST) * 8u, dst = stage_s + static_cast<uint32_t>(st % NST) * (RS * 256u);
            const int site0 = i0 + st * RS * SPW;
            const int n_sites = min(RS * SPW, i1 - site0);                       // sites of the stage that exist
            const uint32_t total = static_cast<uint32_t>(n_sites) * (G * 8u);
            mbar_expect_tx(bar, total);
            const unsigned char *src = row_src + static_cast<size_t>(site0) * R2 * 8u;
            if (R2 == static_cast<uint32_t>(G)) {
                bulk_copy_g2s(dst, src, total, bar);
            } else {      // R > 64: a row is one site's 256 bytes, rows R2 * 8 bytes apart
                for (int k = 0; k < n_sites; ++k) bulk_copy_g2s(dst + k * 256u, src + static_cast<size_t>(k) * R2 * 8u, 256u, bar);
            }
        }
    };
    auto wait_stage = [&](int st) {
        if (st * RS < n_rows) mbar_wait(bar_s + static_cast<uint32_t>(st % NST) * 8u, static_cast<uint32_t>(st / NST) & 1u);
    };
    if constexpr (BULK) {
        if (lane == 0) {
#pragma unroll
            for (int k = 0; k < NST; ++k) mbar_init(bar_s + k * 8u, 1u);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncwarp();
        for (int st = 0; st < NST - 1; ++st) issue_stage(st);
    } else {
        for (int r = 0; r < NS - 1; ++r) issue(std::false_type{}, r);
    }
    auto load_cw = [&](int b) {
        const int i = i0 + b * 32 + lane;
        return i < i1 ? __ldg(co + i) : 0u;
    };
    float2 p1n, p2n;
    uint32_t cw_next = load_cw(1);
    {
        const uint32_t cw0 = load_cw(0);
        p1n = __ldg(a.tab1 + (cw0 & 0xffffu));
        p2n = __ldg(a.tab2 + (cw0 >> 16));
    }
    // one block of 32 sites = RPB rows; FULL: every row read and every row issued by this block exists entirely
    auto block = [&](auto full, int r0) {
        constexpr bool FULL = decltype(full)::value;
        __syncwarp();                                 // the previous block's factors have been read
        fw->fac[lane] = make_float4(p1n.x, p1n.y, p2n.x, p2n.y);
        p1n = __ldg(a.tab1 + (cw_next & 0xffffu));
        p2n = __ldg(a.tab2 + (cw_next >> 16));
        cw_next = load_cw(r0 / RPB + 2);
        __syncwarp();
        constexpr int U = RPB < NS ? RPB : NS;      // unrolled rows: ring slots at compile-time offsets when RPB % NS == 0
#pragma unroll 1
        for (int k0 = 0; k0 < RPB; k0 += U) {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int k = k0 + u;
                const int slot = kConstSlots ? u : (r0 + k) % NS;
                if constexpr (BULK) {
                    if ((kConstSlots ? u : r0 + k) % RS == 0) {      // first row of a stage: refill the stage just read, wait for this one
                        __syncwarp();
                        issue_stage((r0 + k) / RS + NST - 1);
                        wait_stage((r0 + k) / RS);
                    }
                } else {
                    issue(full, (slot + NS - 1) % NS);
                    cp_async_wait<NS - 1>();      // at most NS - 1 younger groups pending: row r0 + k has landed
                }
                if (FULL || (r0 + k < n_rows && i0 + (r0 + k) * SPW + sub < i1))
                    tally(ring_l[slot * 32], fw->fac[k * SPW + sub]);
            }
        }
    };
    int r0 = 0;
    for (; r0 + RPB + NS - 1 <= n_full; r0 += RPB) {
        block(std::true_type{}, r0);
        if ((r0 / RPB) % (256 / RPB) == 256 / RPB - 1) flush();
    }
    for (; r0 < n_rows; r0 += RPB) {
        block(std::false_type{}, r0);
        if ((r0 / RPB) % (256 / RPB) == 256 / RPB - 1) flush();
    }
    if constexpr (!BULK) cp_async_wait<0>();
    unpack();
    __syncthreads();                      // every warp is done with its ring: the space now serves the reduction
    // end of the range: quantise, add the CTA's warps in shared memory (exact integers), one atomic per CTA and sum
    long long (*s_red)[32][16] = reinterpret_cast<long long (*)[32][16]>(f_raw);
#pragma unroll
    for (int c = 0; c < 16; ++c) s_red[warp][lane][c] = __double2ll_rn(static_cast<double>(part[c]) * 4194304.0);
    __syncthreads();
    for (int e = threadIdx.x; e < G * 16; e += blockDim.x) {
        const int ll = e / 16, c = e % 16;
        long long v = 0;
        for (int wi = 0; wi < kWarps; ++wi)
            for (int sb = 0; sb < SPW; ++sb) v += s_red[wi][sb * G + ll][c];
        atomicAdd(reinterpret_cast<unsigned long long *>(a.fk) + (static_cast<size_t>(s) * a.R + 2 * (blockIdx.z * G + ll)) * 8 + c,
                  static_cast<unsigned long long>(v));
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(a.ticket + s, 1u) == gridDim.x * gridDim.z - 1u) ? 1 : 0;
    __syncthreads();
    if (s_last) {
        __threadfence();
        const double inv = 1.0 / 4194304.0;
        for (int r = threadIdx.x; r < a.R; r += blockDim.x) {
            long long *f = a.fk + (static_cast<size_t>(s) * a.R + r) * 8;
            double v[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) { v[c] = static_cast<double>(__ldcg(f + c)) * inv; f[c] = 0; }
            const double g1 = (v[0] * v[0] + v[1] * v[1] + v[2] * v[2] + v[3] * v[3]) / a.N;
            const double g2 = (v[4] * v[4] + v[5] * v[5] + v[6] * v[6] + v[7] * v[7]) / a.N;
            const size_t sr = static_cast<size_t>(s) * a.R + r;
            a.G_slot[2 * sr] = g1;
            a.G_slot[2 * sr + 1] = g2;
            double *o = a.acc_k + (static_cast<size_t>(s) * a.R + a.temp_of_slot[sr]) * 3;
            o[0] += 1.0; o[1] += g1; o[2] += g2;
        }
        if (threadIdx.x == 0) a.ticket[s] = 0u;
    }
}

// ---- random-walk self-return histogram (PAPER.md:149-155 Eq. 11, :436-440 App. A) ------------
// One thread per walker: at step t it jumps to neighbour (x * deg) >> 32 of its site (stays if the site has none), x =
// word (t-1) % 4 of Philox counter (walker, (t-1)/4, sample << 16, domain 4); every visit of its origin at time t adds
// one to hist[sample][t].  Integer work: bit-exact against the oracle.  A step is two dependent random reads (rec,
// col_idx): latency-bound pointer chasing; the walkers of a warp are independent, so the loads of a warp overlap.
// The per-CTA histogram lives in shared memory (32-bit counts), flushed with one 64-bit atomic per time and CTA.
struct WalkArgs {
    const int2 *rec;            // [S][N]
    const int32_t *col_idx;
    const int32_t *start;       // [S][n_walkers]
    unsigned long long *hist;   // [S][n_steps + 1], zero at launch
    int N, n_walkers, n_steps;
    uint32_t sample_base;
    PhiloxKeys keys;
};

__global__ void __launch_bounds__(kBlock) k_random_walk(const WalkArgs a) {
    extern __shared__ unsigned int s_hist[];      // [n_steps + 1]
    const int s = blockIdx.y;
    for (int t = threadIdx.x; t <= a.n_steps; t += blockDim.x) s_hist[t] = 0u;
    __syncthreads();
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w < a.n_walkers) {
        const int2 *rec = a.rec + static_cast<size_t>(s) * a.N;
        const int origin = a.start[static_cast<size_t>(s) * a.n_walkers + w];
        int pos = origin;
        atomicAdd(&s_hist[0], 1u);
        uint32_t x[4] = {0u, 0u, 0u, 0u};
        for (int t = 1; t <= a.n_steps; ++t) {
            const int k = (t - 1) & 3;
            if (k == 0)
                philox4x32_10(static_cast<uint32_t>(w), static_cast<uint32_t>((t - 1) >> 2),
                              (a.sample_base + static_cast<uint32_t>(s)) << 16, kDomWalk, a.keys, x);
            const int2 rc = __ldg(rec + pos);
            const uint32_t deg = static_cast<uint32_t>(rc.y & 0xffff);
            const uint32_t xk = k == 0 ? x[0] : k == 1 ? x[1] : k == 2 ? x[2] : x[3];
            if (deg > 0u) pos = __ldg(a.col_idx + rc.x + static_cast<int>(__umulhi(xk, deg)));
            if (pos == origin) atomicAdd(&s_hist[t], 1u);
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t <= a.n_steps; t += blockDim.x)
        if (s_hist[t]) atomicAdd(a.hist + static_cast<size_t>(s) * (a.n_steps + 1) + t, static_cast<unsigned long long>(s_hist[t]));
}

// ---- acceptance of a Metropolis sweep: angles that differ from the copy taken before it, per (sample, slot) ----
// grid (chunks of sites, samples); a thread owns the slots r = threadIdx.x, + blockDim.x, ... (coalesced rows)
__global__ void __launch_bounds__(kBlock) k_count_changed(const float *before, const float *after, unsigned long long *count,
                                                          int N, int R, int sites_per_block) {
    const int s = blockIdx.y;
    const int i0 = blockIdx.x * sites_per_block, i1 = min(N, i0 + sites_per_block);
    const size_t base = static_cast<size_t>(s) * N * R;
    for (int r = threadIdx.x; r < R; r += blockDim.x) {
        unsigned int c = 0;
        for (int i = i0; i < i1; ++i) {
            const size_t k = base + static_cast<size_t>(i) * R + r;
            c += __float_as_uint(before[k]) != __float_as_uint(after[k]) ? 1u : 0u;
        }
        if (c) atomicAdd(count + static_cast<size_t>(s) * R + r, static_cast<unsigned long long>(c));
    }
}

// ---- init: theta = 2 pi_f * u, Philox domain 0, sweep 0 ------------------------------------------------
__global__ void k_init_theta(float *theta, int S, int N, int R, PhiloxKeys keys, uint32_t sample_base) {
    const size_t total = static_cast<size_t>(S) * N * R;
    for (size_t idx = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; idx < total;
         idx += static_cast<size_t>(gridDim.x) * blockDim.x) {
        const int r = static_cast<int>(idx % R);
        const size_t si = idx / R;
        const int i = static_cast<int>(si % N);
        const int s = static_cast<int>(si / N);
        uint32_t x[4];
        philox4x32_10(static_cast<uint32_t>(i), 0u, ((sample_base + static_cast<uint32_t>(s)) << 16) | static_cast<uint32_t>(r >> 1),
                      kDomInit, keys, x);
        theta[idx] = __fmul_rn(kTwoPiF, (r & 1) ? u01(x[2]) : u01(x[0]));
    }
}

// ---- stand-alone swap round (one CTA per sample), counters, labels -> per-slot parameters ----
__global__ void k_pt_swap(const SwapArgs a) { pt_swap_sample(a, blockIdx.x, a.counters[1]); }

__global__ void k_tick(uint32_t *counters, uint32_t d_sweep, uint32_t d_round) {
    counters[0] += d_sweep;
    counters[1] += d_round;
}

// labels -> per-slot parameters (after xy_set_labels)
__global__ void k_refresh_slot_params(const int32_t *temp_of_slot, int32_t *slot_of_temp, const float *beta_f,
                                      const float *w_f, float *beta_slot, float *w_slot, int S, int R) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= S * R) return;
    const int s = idx / R, t = temp_of_slot[idx];
    slot_of_temp[static_cast<size_t>(s) * R + t] = idx % R;
    beta_slot[idx] = beta_f[t];
    w_slot[idx] = w_f[t];
}

}  // namespace xy
