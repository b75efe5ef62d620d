// xy_kernels.cuh -- sm_100a kernels of the XY / Levy-graph hot path (see include/xy_b200.h).
//
// Layout: theta[S][N][R] fp32, replica (slot) fastest.  A lane owns TWO adjacent slots (one float2 and
// one Philox4x32-10 call per site: words (x0,x1) feed the even slot, (x2,x3) the odd one), so a group of
// G = R/2 lanes covers one site and a warp covers 32/G sites.  At R = 64 a warp gathers one neighbour as
// one 256-byte coalesced request.  The neighbour ids of a site are fetched with ONE coalesced load
// (lane l takes col_idx[start + l]) and broadcast with shuffles.
//
// PAPER.md:444,:454 (coloured single-spin Metropolis), :460 (over-relaxation, ref 66), :167-181 (E, m),
// :460-472 (parallel tempering); readings R5-R11 in DESIGN.md.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace xy {

constexpr float kTwoPiF = 6.2831855f;           // fp32(2 pi)
constexpr float kTwoPiLo = -1.7484555e-7f;      // 2 pi - fp32(2 pi)
constexpr float kInvTwoPiF = 0.15915494f;
constexpr unsigned kFull = 0xffffffffu;
constexpr int kBlock = 256;                     // threads per CTA in the class kernels
constexpr int kWarps = kBlock / 32;

enum : uint32_t { kDomInit = 0u, kDomMetropolis = 1u, kDomSwap = 2u };

// ---- Philox4x32-10 (Salmon et al., SC'11), written from the round function -------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t (&x)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = static_cast<unsigned long long>(0xD2511F53u) * c0;
        const unsigned long long p1 = static_cast<unsigned long long>(0xCD9E8D57u) * c2;
        const uint32_t n0 = static_cast<uint32_t>(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = static_cast<uint32_t>(p0 >> 32) ^ c3 ^ k1;
        c1 = static_cast<uint32_t>(p1);
        c3 = static_cast<uint32_t>(p0);
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    x[0] = c0; x[1] = c1; x[2] = c2; x[3] = c3;
}

// u = ((x >> 9) + 0.5) 2^-23: every step exact in fp32 (R11)
__device__ __forceinline__ float u01(uint32_t x) {
    return fmaf(static_cast<float>(x >> 9), 1.1920928955078125e-07f, 5.9604644775390625e-08f);
}

// ---- arguments shared by the per-colour kernels ------------------------------------------------------
struct ClassArgs {
    const int2 *rec;           // [S][N] {first col_idx entry (absolute), degree}
    const int32_t *col_idx;    // concatenated neighbour ids (local to the sample)
    const int32_t *class_ptr;  // [S][q_stride]
    float *theta;              // [S][N][R]
    const float *beta_slot;    // [S][R]
    const float *w_slot;       // [S][R]
    const uint32_t *counters;  // device {sweep, round}
    int N, R, q_stride, colour, s0, chunk;  // chunk = site groups per warp
    uint32_t sweep_fixed;
    int sweep_offset, use_counter;
    uint32_t key0, key1, sample_base;
};

// Metropolis for one slot given the sum over neighbours of sin(mid - theta_j):
//   dE = -sum_j[cos(th' - th_j) - cos(th - th_j)] = 2 sin((th'-th)/2) sum_j sin((th'+th)/2 - th_j)
__device__ __forceinline__ float metropolis_finish(float own, float thp, float half, float ssum, float beta,
                                                   float u2) {
    const float dE = 2.0f * __sinf(half) * ssum;
    const float p = __expf(-beta * dE);
    float wrapped = thp;
    if (thp >= kTwoPiF) wrapped = thp - kTwoPiF;
    else if (thp < 0.0f) wrapped = thp + kTwoPiF;
    return (u2 < p) ? wrapped : own;
}

// over-relaxation for one slot given the local field h (R7)
__device__ __forceinline__ float overrelax_finish(float own, float hx, float hy) {
    if (hx == 0.0f && hy == 0.0f) return own;
    float t = 2.0f * atan2f(hy, hx) - own;                 // in [-4 pi, 2 pi]
    const float k = floorf(t * kInvTwoPiF);
    t = fmaf(-k, kTwoPiF, t);
    t = fmaf(-k, kTwoPiLo, t);
    if (t < 0.0f) t += kTwoPiF;
    if (t >= kTwoPiF) t -= kTwoPiF;
    return t;
}

// ---- fast path: R = 2 G (G a power of two <= 32) or R a multiple of 64 (G = 32, blockIdx.z = column block)
// MODE 0 = Metropolis, 1 = over-relaxation.
template <int G, int MODE>
__global__ void __launch_bounds__(kBlock) k_update_class(const ClassArgs a) {
    constexpr int SPW = 32 / G;              // sites per warp
    constexpr int UNR = G < 8 ? G : 8;       // neighbour gathers issued back to back
    const int s = a.s0 + blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sub = lane / G, l = lane % G;
    const int R2 = a.R >> 1;
    const int q = blockIdx.z * G + l;        // slot pair handled by this lane

    const int cbeg = a.class_ptr[s * a.q_stride + a.colour];
    const int cend = a.class_ptr[s * a.q_stride + a.colour + 1];
    const int n_groups = (cend - cbeg + SPW - 1) / SPW;
    const int g0 = (blockIdx.x * kWarps + warp) * a.chunk;
    if (g0 >= n_groups) return;
    const int g1 = min(g0 + a.chunk, n_groups);

    float2 *__restrict__ th2 = reinterpret_cast<float2 *>(a.theta) + static_cast<size_t>(s) * a.N * R2;
    const int2 *__restrict__ rec = a.rec + static_cast<size_t>(s) * a.N;

    float2 beta = make_float2(0.f, 0.f), w = make_float2(0.f, 0.f);
    uint32_t sweep = 0, c2 = 0;
    if (MODE == 0) {
        beta = reinterpret_cast<const float2 *>(a.beta_slot)[static_cast<size_t>(s) * R2 + q];
        w = reinterpret_cast<const float2 *>(a.w_slot)[static_cast<size_t>(s) * R2 + q];
        sweep = a.use_counter ? a.counters[0] + static_cast<uint32_t>(a.sweep_offset) : a.sweep_fixed;
        c2 = ((a.sample_base + static_cast<uint32_t>(s)) << 16) | static_cast<uint32_t>(q);
    }

    for (int g = g0; g < g1; ++g) {
        const int i = cbeg + g * SPW + sub;
        const bool valid = i < cend;
        int2 rc = make_int2(0, 0);
        if (valid) rc = rec[i];
        const int deg = rc.y;
        const int degmax = (SPW == 1) ? deg : __reduce_max_sync(kFull, deg);
        float2 own = make_float2(0.f, 0.f);
        if (valid) own = th2[static_cast<size_t>(i) * R2 + q];

        // per-slot state: Metropolis (mid-angle, half-step, sum of sines) or OR (hx, hy)
        float midx = 0.f, midy = 0.f, halfx = 0.f, halfy = 0.f, thpx = 0.f, thpy = 0.f;
        float u2x = 0.f, u2y = 0.f;
        float ax = 0.f, ay = 0.f, bx = 0.f, by = 0.f;   // MET: ax, ay = sine sums; OR: (ax,bx) = h of .x slot
        if (MODE == 0) {
            uint32_t x[4];
            philox4x32_10(static_cast<uint32_t>(i), sweep, c2, kDomMetropolis, a.key0, a.key1, x);
            const float dx = __fmul_rn(w.x, u01(x[0]) - 0.5f);
            const float dy = __fmul_rn(w.y, u01(x[2]) - 0.5f);
            u2x = u01(x[1]);
            u2y = u01(x[3]);
            thpx = __fadd_rn(own.x, dx);
            thpy = __fadd_rn(own.y, dy);
            halfx = 0.5f * (thpx - own.x);
            halfy = 0.5f * (thpy - own.y);
            midx = own.x + halfx;
            midy = own.y + halfy;
        }

        for (int base = 0; base < degmax; base += G) {
            int myidx = -1;
            if (base + l < deg) myidx = a.col_idx[rc.x + base + l];
#pragma unroll 1
            for (int k0 = 0; k0 < G && base + k0 < degmax; k0 += UNR) {
                float2 t[UNR];
                bool ok[UNR];
#pragma unroll
                for (int u = 0; u < UNR; ++u) {
                    const int j = __shfl_sync(kFull, myidx, k0 + u, G);
                    ok[u] = j >= 0;
                    t[u] = make_float2(0.f, 0.f);
                    if (ok[u]) t[u] = th2[static_cast<size_t>(j) * R2 + q];
                }
#pragma unroll
                for (int u = 0; u < UNR; ++u) {
                    if (ok[u]) {
                        if (MODE == 0) {
                            ax += __sinf(midx - t[u].x);
                            ay += __sinf(midy - t[u].y);
                        } else {
                            float sn, cs;
                            __sincosf(t[u].x, &sn, &cs);
                            ax += cs; bx += sn;
                            __sincosf(t[u].y, &sn, &cs);
                            ay += cs; by += sn;
                        }
                    }
                }
            }
        }

        if (valid) {
            float2 out;
            if (MODE == 0) {
                out.x = metropolis_finish(own.x, thpx, halfx, ax, beta.x, u2x);
                out.y = metropolis_finish(own.y, thpy, halfy, ay, beta.y, u2y);
            } else {
                out.x = overrelax_finish(own.x, ax, bx);
                out.y = overrelax_finish(own.y, ay, by);
            }
            th2[static_cast<size_t>(i) * R2 + q] = out;
        }
    }
}

// ---- generic path: any R >= 1 (odd R, R = 6, ...): one warp per site, lanes stride over the slots ----
template <int MODE>
__global__ void __launch_bounds__(kBlock) k_update_class_generic(const ClassArgs a) {
    const int s = a.s0 + blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int cbeg = a.class_ptr[s * a.q_stride + a.colour];
    const int cend = a.class_ptr[s * a.q_stride + a.colour + 1];
    const int n_sites = cend - cbeg;
    const int g0 = (blockIdx.x * kWarps + warp) * a.chunk;
    if (g0 >= n_sites) return;
    const int g1 = min(g0 + a.chunk, n_sites);
    float *__restrict__ th = a.theta + static_cast<size_t>(s) * a.N * a.R;
    const int2 *__restrict__ rec = a.rec + static_cast<size_t>(s) * a.N;
    const uint32_t sweep = a.use_counter ? a.counters[0] + static_cast<uint32_t>(a.sweep_offset) : a.sweep_fixed;

    for (int g = g0; g < g1; ++g) {
        const int i = cbeg + g;
        const int2 rc = rec[i];
        for (int r = lane; r < a.R; r += 32) {
            const float own = th[static_cast<size_t>(i) * a.R + r];
            float thp = 0.f, half = 0.f, mid = 0.f, u2 = 0.f, acc0 = 0.f, acc1 = 0.f;
            if (MODE == 0) {
                uint32_t x[4];
                philox4x32_10(static_cast<uint32_t>(i), sweep,
                              ((a.sample_base + static_cast<uint32_t>(s)) << 16) | static_cast<uint32_t>(r >> 1),
                              kDomMetropolis, a.key0, a.key1, x);
                const float u1 = (r & 1) ? u01(x[2]) : u01(x[0]);
                u2 = (r & 1) ? u01(x[3]) : u01(x[1]);
                const float w = a.w_slot[static_cast<size_t>(s) * a.R + r];
                thp = __fadd_rn(own, __fmul_rn(w, u1 - 0.5f));
                half = 0.5f * (thp - own);
                mid = own + half;
            }
            for (int e = 0; e < rc.y; ++e) {
                const float t = th[static_cast<size_t>(a.col_idx[rc.x + e]) * a.R + r];
                if (MODE == 0) {
                    acc0 += __sinf(mid - t);
                } else {
                    float sn, cs;
                    __sincosf(t, &sn, &cs);
                    acc0 += cs; acc1 += sn;
                }
            }
            float out;
            if (MODE == 0)
                out = metropolis_finish(own, thp, half, acc0, a.beta_slot[static_cast<size_t>(s) * a.R + r], u2);
            else
                out = overrelax_finish(own, acc0, acc1);
            th[static_cast<size_t>(i) * a.R + r] = out;
        }
    }
}

// ---- init: theta = 2 pi_f * u, Philox domain 0, sweep 0 ------------------------------------------------
__global__ void k_init_theta(float *theta, int S, int N, int R, uint32_t key0, uint32_t key1,
                             uint32_t sample_base) {
    const size_t total = static_cast<size_t>(S) * N * R;
    for (size_t idx = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; idx < total;
         idx += static_cast<size_t>(gridDim.x) * blockDim.x) {
        const int r = static_cast<int>(idx % R);
        const size_t si = idx / R;
        const int i = static_cast<int>(si % N);
        const int s = static_cast<int>(si / N);
        uint32_t x[4];
        philox4x32_10(static_cast<uint32_t>(i), 0u, ((sample_base + static_cast<uint32_t>(s)) << 16) | static_cast<uint32_t>(r >> 1),
                      kDomInit, key0, key1, x);
        theta[idx] = __fmul_rn(kTwoPiF, (r & 1) ? u01(x[2]) : u01(x[0]));
    }
}

// ---- measure: E = -sum_{i<j} cos(theta_i - theta_j), M = sum_i (cos, sin) per slot ---------------------
// grid (n_chunks, samples in group); each CTA reduces a contiguous range of `chunk_sites` sites of one
// sample and writes partial[s][chunk][r][3] (fp64).  Fixed summation order -> bit-reproducible.
struct MeasureArgs {
    const int2 *rec;
    const int32_t *col_idx;
    const float *theta;
    double *partial;   // [S][n_chunks][R][3]
    int N, R, s0, n_chunks, chunk_sites;
};

__global__ void __launch_bounds__(kBlock) k_measure_partial(const MeasureArgs a) {
    extern __shared__ double sm[];   // [kWarps][R][3]
    const int s = a.s0 + blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ibeg = blockIdx.x * a.chunk_sites;
    const int iend = min(ibeg + a.chunk_sites, a.N);
    const float *__restrict__ th = a.theta + static_cast<size_t>(s) * a.N * a.R;
    const int2 *__restrict__ rec = a.rec + static_cast<size_t>(s) * a.N;

    for (int r0 = 0; r0 < a.R; r0 += 32) {
        const int r = r0 + lane;
        double e = 0.0, mx = 0.0, my = 0.0;
        if (r < a.R) {
            for (int i = ibeg + warp; i < iend; i += kWarps) {
                const int2 rc = rec[i];
                const float own = th[static_cast<size_t>(i) * a.R + r];
                float sn, cs;
                sincosf(own, &sn, &cs);
                mx += static_cast<double>(cs);
                my += static_cast<double>(sn);
                float esite = 0.f;
                for (int q = 0; q < rc.y; ++q) {
                    const int j = a.col_idx[rc.x + q];
                    if (j > i) esite += cosf(own - th[static_cast<size_t>(j) * a.R + r]);
                }
                e -= static_cast<double>(esite);
            }
            double *row = sm + (static_cast<size_t>(warp) * a.R + r) * 3;
            row[0] = e; row[1] = mx; row[2] = my;
        }
    }
    __syncthreads();
    double *out = a.partial + (static_cast<size_t>(s) * a.n_chunks + blockIdx.x) * a.R * 3;
    for (int idx = threadIdx.x; idx < a.R * 3; idx += kBlock) {
        double acc = 0.0;
        for (int wi = 0; wi < kWarps; ++wi) acc += sm[static_cast<size_t>(wi) * a.R * 3 + idx];
        out[idx] = acc;
    }
}

// one thread per (sample, slot): sum the chunk partials in order, publish E/M per slot and (optionally)
// add Eq. 13-16 moments to the accumulators of the slot's temperature.
__global__ void k_measure_final(const double *partial, int s0, int s1, int N, int R, int n_chunks,
                                const int32_t *temp_of_slot, double *E_slot, double *M_slot, double *acc,
                                int accumulate) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    const int s = s0 + idx / R, r = idx % R;
    if (s >= s1) return;
    double e = 0.0, mx = 0.0, my = 0.0;
    for (int c = 0; c < n_chunks; ++c) {
        const double *p = partial + ((static_cast<size_t>(s) * n_chunks + c) * R + r) * 3;
        e += p[0]; mx += p[1]; my += p[2];
    }
    E_slot[static_cast<size_t>(s) * R + r] = e;
    M_slot[(static_cast<size_t>(s) * R + r) * 2] = mx;
    M_slot[(static_cast<size_t>(s) * R + r) * 2 + 1] = my;
    if (accumulate) {
        double *a = acc + (static_cast<size_t>(s) * R + temp_of_slot[static_cast<size_t>(s) * R + r]) * 8;
        const double ux = mx / N, uy = my / N, m2 = ux * ux + uy * uy;
        a[0] += 1.0; a[1] += e; a[2] += e * e; a[3] += sqrt(m2); a[4] += m2; a[5] += m2 * m2;
        a[6] += ux; a[7] += uy;
    }
}

// ---- parallel-tempering swap round: one CTA per sample -------------------------------------------------
struct SwapArgs {
    const double *E_slot;       // [S][R]
    const double *betaT;        // [R] 1/T fp64
    const float *beta_f;        // [R]
    const float *w_f;           // [R]
    int32_t *slot_of_temp;      // [S][R]
    int32_t *temp_of_slot;      // [S][R]
    float *beta_slot, *w_slot;  // [S][R]
    const uint32_t *counters;
    const uint8_t *decisions;   // [S][R] or nullptr
    long long *attempts, *accepts;  // [S][R]
    int R;
    uint32_t key0, key1, sample_base;
};

__global__ void k_pt_swap(const SwapArgs a) {
    const int s = blockIdx.x;
    const uint32_t round = a.counters[1];
    const int parity = static_cast<int>(round & 1u);
    int32_t *sot = a.slot_of_temp + static_cast<size_t>(s) * a.R;
    int32_t *tos = a.temp_of_slot + static_cast<size_t>(s) * a.R;
    for (int t = parity + 2 * static_cast<int>(threadIdx.x); t + 1 < a.R; t += 2 * blockDim.x) {
        const int sa = sot[t], sb = sot[t + 1];
        bool acc;
        if (a.decisions) {
            acc = a.decisions[static_cast<size_t>(s) * a.R + t] != 0;
        } else {
            uint32_t x[4];
            philox4x32_10(static_cast<uint32_t>(t), round, (a.sample_base + static_cast<uint32_t>(s)) << 16, kDomSwap,
                          a.key0, a.key1, x);
            const double u = static_cast<double>(u01(x[0]));
            const double arg = (a.betaT[t] - a.betaT[t + 1]) *
                               (a.E_slot[static_cast<size_t>(s) * a.R + sa] - a.E_slot[static_cast<size_t>(s) * a.R + sb]);
            acc = u < exp(arg);
        }
        a.attempts[static_cast<size_t>(s) * a.R + t] += 1;
        if (acc) {
            a.accepts[static_cast<size_t>(s) * a.R + t] += 1;
            sot[t] = sb; sot[t + 1] = sa;
            tos[sa] = t + 1; tos[sb] = t;
        }
    }
    __syncthreads();
    for (int r = threadIdx.x; r < a.R; r += blockDim.x) {
        const int t = tos[r];
        a.beta_slot[static_cast<size_t>(s) * a.R + r] = a.beta_f[t];
        a.w_slot[static_cast<size_t>(s) * a.R + r] = a.w_f[t];
    }
}

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
