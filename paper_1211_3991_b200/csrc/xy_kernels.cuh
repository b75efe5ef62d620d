// xy_kernels.cuh -- shared device pieces of the XY / Levy-graph hot path (see include/xy_b200.h):
// Philox4x32-10, the Metropolis / over-relaxation finishing arithmetic, the kernel argument blocks and the swap round.
// The product path for R = 2 * 2^k <= 64 and R % 64 == 0 is k_phase (one launch per colour class, xy_sweep.cuh) and,
// for small samples, k_cycle (one cluster per sample, xy_cycle.cuh); the small kernels and the any-R path are in
// xy_aux_kernels.cuh.
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
constexpr int kBlock = 256;                     // threads per CTA
constexpr int kWarps = kBlock / 32;
constexpr double kFix = 68719476736.0;          // 2^36: fixed-point scale of the measure reduction
constexpr double kInvFix = 1.0 / 68719476736.0;

enum : uint32_t { kDomInit = 0u, kDomMetropolis = 1u, kDomSwap = 2u, kDomWalk = 4u };
enum : int { kModeMetropolis = 0, kModeOverrelax = 1, kModeMeasure = 2, kModeOrMeasure = 3, kModeMetOr = 4, kModeMetOrMeasure = 5 };

// ---- Philox4x32-10 (Salmon et al., SC'11), written from the round function -------------------------
// ks[2r], ks[2r+1] = the round keys k0 + r W0, k1 + r W1 (W0 = 0x9E3779B9, W1 = 0xBB67AE85)
struct PhiloxKeys { uint32_t ks[20]; };

__host__ __device__ inline PhiloxKeys philox_key_schedule(uint32_t k0, uint32_t k1) {
    PhiloxKeys k;
    for (int r = 0; r < 10; ++r) {
        k.ks[2 * r] = k0;
        k.ks[2 * r + 1] = k1;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return k;
}

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              const PhiloxKeys &k, uint32_t (&x)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = static_cast<unsigned long long>(0xD2511F53u) * c0;
        const unsigned long long p1 = static_cast<unsigned long long>(0xCD9E8D57u) * c2;
        const uint32_t n0 = static_cast<uint32_t>(p1 >> 32) ^ c1 ^ k.ks[2 * r];
        const uint32_t n2 = static_cast<uint32_t>(p0 >> 32) ^ c3 ^ k.ks[2 * r + 1];
        c1 = static_cast<uint32_t>(p1);
        c3 = static_cast<uint32_t>(p0);
        c0 = n0;
        c2 = n2;
    }
    x[0] = c0; x[1] = c1; x[2] = c2; x[3] = c3;
}

// u = ((x >> 9) + 0.5) 2^-23: every step exact in fp32 (R11)
__device__ __forceinline__ float u01(uint32_t x) {
    return fmaf(static_cast<float>(x >> 9), 1.1920928955078125e-07f, 5.9604644775390625e-08f);
}

// ---- cp.async (LDGSTS): 8 bytes per lane, global -> shared, no register staging ---------------------------
__device__ __forceinline__ void cp_async8(uint32_t smem_addr, const void *gptr) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_addr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- arguments shared by the update / measure kernels -----------------------------------------------------------------
struct TileArgs {
    const int2 *rec;           // [S][N] {first col_idx entry (absolute), degree | n_lower << 16}
    const int32_t *col_idx;    // concatenated neighbour ids (local to the sample), ascending per site
    const int32_t *class_ptr;  // [S][q_stride]
    float *theta;              // [S][N][R]
    const float *beta_slot;    // [S][R]
    const float *w_slot;       // [S][R]
    const uint32_t *counters;  // device {sweep, round}
    int N, R, q_stride, colour, s0, tiles_per_warp;
    uint32_t sweep_fixed;
    int sweep_offset, use_counter;
    uint32_t sample_base;
    PhiloxKeys keys;
    // measure only
    long long *fx;             // [2][S][R][3] fixed-point sums (E, Mx, My), zero between launches (k_phase uses buffer 0)
    size_t fx_stride;          // S * R * 3: offset of the second buffer
    unsigned int *ticket;      // [S] CTAs done, zero between launches
    const int32_t *temp_of_slot;
    double *E_slot, *M_slot, *acc;
    int accumulate;
};

// wrap the proposal once by +-2 pi_f (R5) and keep it iff u2 < p (R6, strict)
__device__ __forceinline__ float metropolis_select(float own, float thp, float u2, float p) {
    float wrapped = thp;
    if (thp >= kTwoPiF) wrapped = thp - kTwoPiF;
    else if (thp < 0.0f) wrapped = thp + kTwoPiF;
    return (u2 < p) ? wrapped : own;
}

// atan2(y, x) for (x, y) != (0, 0): octant reduction, a = min/max in [0, 1] by MUFU.RCP, odd minimax polynomial
// a P(a^2) with 8 coefficients (max abs error 1.3e-7 rad in fp32 arithmetic, i.e. about one ulp of pi/4; the
// error budget of R7 is 5e-6).  About 25 instructions instead of the ~60 of atan2f.
__device__ __forceinline__ float fast_atan2(float y, float x) {
    const float ax = fabsf(x), ay = fabsf(y);
    const float a = __fdividef(fminf(ax, ay), fmaxf(ax, ay));
    const float s = a * a;
    float p = -0.004054560326039791f;
    p = fmaf(p, s, 0.021862933412194252f);
    p = fmaf(p, s, -0.05591229349374771f);
    p = fmaf(p, s, 0.09642194956541061f);
    p = fmaf(p, s, -0.1390862911939621f);
    p = fmaf(p, s, 0.19946566224098206f);
    p = fmaf(p, s, -0.33329859375953674f);
    p = fmaf(p, s, 0.9999993443489075f);
    float r = p * a;
    if (ay > ax) r = 1.5707963267948966f - r;
    if (x < 0.0f) r = 3.14159265358979f - r;
    return copysignf(r, y);
}

// over-relaxation for one slot given the local field h (R7)
__device__ __forceinline__ float overrelax_finish(float own, float hx, float hy) {
    if (hx == 0.0f && hy == 0.0f) return own;
    float t = 2.0f * fast_atan2(hy, hx) - own;             // in [-4 pi, 2 pi]
    const float k = floorf(t * kInvTwoPiF);
    t = fmaf(-k, kTwoPiF, t);
    t = fmaf(-k, kTwoPiLo, t);
    if (t < 0.0f) t += kTwoPiF;
    if (t >= kTwoPiF) t -= kTwoPiF;
    return t;
}

// ---- parallel-tempering swap round: one CTA per sample ----
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
    PhiloxKeys keys;
    uint32_t sample_base;
};

// one swap round of sample s by the calling CTA (all its threads; ends with a __syncthreads-separated refresh of the
// per-slot parameters): pairs (t, t+1), t = round mod 2 (mod 2); accept iff u < exp((beta_t - beta_t+1)(E_a - E_b)) (R9)
__device__ __forceinline__ void pt_swap_sample(const SwapArgs &a, int s, uint32_t round) {
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
                          a.keys, x);
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

}  // namespace xy
