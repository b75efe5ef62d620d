// xy_b200.cu -- C-ABI implementation (include/xy_b200.h): handles, validation, launches, CUDA graphs.
// Every step of the hot path runs in the kernels of xy_kernels.cuh; nothing here computes physics.
#include "xy_b200.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <tuple>
#include <vector>

#include "xy_aux_kernels.cuh"
#include "xy_cycle.cuh"
#include "xy_diag.cuh"
#include "xy_dispatch.h"
#include "xy_kernels.cuh"
#include "xy_sweep.cuh"

namespace {

thread_local std::string g_err;
thread_local double g_walk_kernel_us = -1.0;      // device time of the calling thread's last k_random_walk launch

int fail(int code, const std::string &msg) {
    g_err = msg;
    return code;
}

#define XY_CUDA(call)                                                                              \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(XY_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));             \
    } while (0)

template <typename T>
int dev_alloc(T **p, size_t n) {
    *p = nullptr;
    if (n == 0) n = 1;
    cudaError_t e = cudaMalloc(reinterpret_cast<void **>(p), n * sizeof(T));
    if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? XY_ENOMEM : XY_ECUDA,
                                      std::string("cudaMalloc: ") + cudaGetErrorString(e));
    return XY_OK;
}

int ceil_div(long long a, long long b) { return static_cast<int>((a + b - 1) / b); }

// persisting-L2 carve-out: raised while at least one ensemble lives on the device, put back by the last xy_pt_destroy
std::mutex g_l2_mutex;
std::map<int, std::pair<int, size_t>> g_l2_users;      // device -> (live ensembles, limit found before the first one)

bool l2_carveout_acquire(int dev, size_t bytes) {
    std::lock_guard<std::mutex> lock(g_l2_mutex);
    auto &u = g_l2_users[dev];
    if (u.first == 0) {
        size_t before = 0;
        if (cudaDeviceGetLimit(&before, cudaLimitPersistingL2CacheSize) != cudaSuccess ||
            cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, bytes) != cudaSuccess) {
            cudaGetLastError();
            return false;
        }
        u.second = before;
    }
    u.first += 1;
    return true;
}

void l2_carveout_release(int dev) {
    std::lock_guard<std::mutex> lock(g_l2_mutex);
    auto it = g_l2_users.find(dev);
    if (it == g_l2_users.end() || it->second.first == 0) return;
    if (--it->second.first == 0) {
        cudaCtxResetPersistingL2Cache();
        cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, it->second.second);
        cudaGetLastError();
    }
}

// every entry point runs on the device its handle was created on and leaves the caller's current device unchanged
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev) {
        if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};

}  // namespace

namespace xy {

const void *phase_function(int W, int G, bool single_block, int mode) {
    if (W == 24 || W == 28) return phase_function_w24(G, single_block, mode);      // the measuring modes' own CTA shapes
    if (W == kWarpsSmall) return mode < 3 ? phase_function_w8_a(G, single_block, mode) : phase_function_w8_b(G, single_block, mode);
    if (W == kWarpsBig) return mode < 3 ? phase_function_w32_a(G, single_block, mode) : phase_function_w32_b(G, single_block, mode);
    return nullptr;
}

const void *cycle_function(int order, int G) { return order == 0 ? cycle_function_o0(G) : cycle_function_o1(G); }

}  // namespace xy

struct xy_graph {
    int S = 0, N = 0, q_max = 0, q_stride = 0, max_degree = 0;
    long long nnz_total = 0;
    int2 *rec = nullptr;
    int32_t *col_idx = nullptr;
    int32_t *class_ptr = nullptr;
    std::vector<int32_t> h_class_ptr;  // [S][q_stride]
    std::vector<uint32_t> h_deg;       // [S][N] degree | n_lower << 16 (host copy of rec.y, for the share tables)
    std::vector<long long> h_off;      // [S+1] first col_idx entry of every sample
    size_t bytes_per_sample = 0;       // rec + col_idx (average), for the schedule heuristic
    int Lx = 0, Ly = 0;                // lattice extents of the site coordinates (0 = none set)
    uint32_t *coords = nullptr;        // [S][N] x | y << 16
    float2 *tab1 = nullptr, *tab2 = nullptr;   // [Lx], [Ly]: (cos, sin)(2 pi n / L)
    cudaStream_t stream = nullptr;
    int device = -1, n_sm = 0;         // the CUDA device the graph lives on (current device of xy_graph_load)
};

struct CycleKey {
    int sps, orps, me, phase, group, await_upload;
    bool operator<(const CycleKey &o) const {
        return std::tie(sps, orps, me, phase, group, await_upload) < std::tie(o.sps, o.orps, o.me, o.phase, o.group, o.await_upload);
    }
};

struct CycleGraph {
    cudaGraphExec_t exec = nullptr;
    long long launches = 0;
};

struct xy_pt {
    const xy_graph *g = nullptr;
    int R = 0;
    uint32_t key0 = 0, key1 = 0, sample_base = 0;
    cudaStream_t stream = nullptr;
    bool owns_stream = false;
    float *theta = nullptr;
    bool owns_theta = false;
    float *beta_slot = nullptr, *w_slot = nullptr, *beta_f = nullptr, *w_f = nullptr;
    double *betaT = nullptr;
    int32_t *temp_of_slot = nullptr, *slot_of_temp = nullptr;
    uint32_t *counters = nullptr;
    double *E_slot = nullptr, *M_slot = nullptr, *acc = nullptr;
    double *G_slot = nullptr, *acc_k = nullptr;   // structure factor at k_min: [S][R][2] per slot, [S][R][3] by temperature
    long long *fk = nullptr;                      // [S][R][8] fixed-point sums of k_fourier
    long long *fx = nullptr;            // [S][R][3] fixed-point measure sums (zero between launches)
    unsigned int *ticket = nullptr;     // [S]
    long long *attempts = nullptr, *accepts = nullptr;
    uint8_t *decisions = nullptr;
    xy::PhiloxKeys keys;
    int fast_G = 0;  // lanes per site of the float2 kernel (k_phase), 0 = any-R kernels
    int col_blocks = 1;
    int l2_persist = 1;              // mark the running sample group's theta as persisting in L2 (access policy window)
    size_t l2_persist_bytes = 0, l2_window_max = 0;   // device limits (0 = not supported)
    bool l2_limit_set = false;       // this ensemble holds a reference on the device's persisting-L2 carve-out
    int balance = 1;                 // cost-balanced share tables (1) or equal shares (0)
    int pdl = 1;                     // programmatic dependent launch edges between the k_phase launches
    const void *phase_fn[2][6] = {};   // k_phase<G, CB, MODE, W>: [0] W = 8 warps per CTA, [1] W = 32
    const void *phase_fn24[2] = {nullptr, nullptr};   // measuring modes 3 (28-warp CTAs, 72 registers) and 5 (24-warp CTAs, 80): no spills
    int order = 0;                   // 0 = Metropolis sweep then OR sweep, 1 = interleaved by colour (xy_set_order)
    int capacity_big = 0;            // co-resident 32-warp CTAs (one per SM)
    int cta_shape = 0;               // 0 = by class size, 1 = always 8-warp CTAs, 2 = always 32-warp CTAs
    int path = 0;                    // xy_set_path: 0 = automatic, 1 = one launch per colour class (k_phase), 2 = one cluster per sample (k_cycle)
    const void *cycle_fn[2] = {nullptr, nullptr};   // k_cycle<G, ORDER>, by order
    int cycle_smem_max = 0;          // largest dynamic shared memory of a k_cycle CTA on this device (0 = cluster path not available)
    int cycle_C_max = 8;             // largest cluster size tried: 16 when the device allows the non-portable size
    // the plan of the cluster path (cycle_plan; made at the first use): CTAs per sample, per-warp resident pool
    int cycle_planned = 0;           // 0 = not yet, 1 = planned, -1 = the samples do not fit
    int cycle_C = 0, cycle_k_cap = 0, cycle_id_cap = 0, cycle_resident = 0;
    int fuse_measure = 1;            // measured sweeps: the last over-relaxation sweep also produces E, Mx, My (MODE 3)
    std::map<int, int4 *> parts;     // warps per sample -> device [S][q_stride][nw] share tables {i0, w1, start0, n_run}
    int sweep_capacity = 0;          // co-resident CTAs of k_phase on this device: the grid is one such wave
    int measure_chunk = 256;  // sites per CTA of the generic measure kernel
    int samples_per_group = 0;  // 0 = automatic
    // host mirrors
    uint32_t sweep = 0, round = 0;
    bool e_fresh = false;
    long long launches = 0;
    std::map<CycleKey, CycleGraph> graphs;
    // xy_set_theta_async: group-wise uploads on a second stream, awaited group by group inside the next cycle
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t compute_done = nullptr;
    std::vector<cudaEvent_t> upload_ev;   // one per sample group of the schedule the upload was issued for
    int upload_group = 0;                 // samples per group of that schedule
    bool upload_armed = false;            // uploads in flight that the compute stream has not been ordered after yet
};

namespace {

// ------------------------------------------------------------------------------------------------
// launches
// ------------------------------------------------------------------------------------------------
int max_class_size(const xy_graph *g, int colour, int s0, int s1) {
    int m = 0;
    for (int s = s0; s < s1; ++s) {
        const int32_t *cp = g->h_class_ptr.data() + static_cast<size_t>(s) * g->q_stride;
        m = std::max(m, cp[colour + 1] - cp[colour]);
    }
    return m;
}

xy::TileArgs tile_args(const xy_pt *pt, int colour, int s0) {
    const xy_graph *g = pt->g;
    xy::TileArgs a;
    a.rec = g->rec; a.col_idx = g->col_idx; a.class_ptr = g->class_ptr; a.theta = pt->theta;
    a.beta_slot = pt->beta_slot; a.w_slot = pt->w_slot; a.counters = pt->counters;
    a.N = g->N; a.R = pt->R; a.q_stride = g->q_stride; a.colour = colour; a.s0 = s0; a.tiles_per_warp = 1;
    a.sweep_fixed = 0u; a.sweep_offset = 0; a.use_counter = 0;
    a.sample_base = pt->sample_base; a.keys = pt->keys;
    a.fx = pt->fx; a.fx_stride = static_cast<size_t>(g->S) * pt->R * 3; a.ticket = pt->ticket; a.temp_of_slot = pt->temp_of_slot;
    a.E_slot = pt->E_slot; a.M_slot = pt->M_slot; a.acc = pt->acc; a.accumulate = 0;
    return a;
}

// ---- share tables: for nw warps per sample, the first site of every warp's contiguous share of each colour class
// (and, at colour index q_max, of the measure pass over all sites), balanced by cost = const + degree.  Integer
// bookkeeping only; the kernels give the same results for any partition (sites of a class are independent, the
// measure sums are exact integers). ----
int get_partition(xy_pt *pt, int nw, const int4 **out) {
    auto it = pt->parts.find(nw);
    if (it != pt->parts.end()) { *out = it->second; return XY_OK; }
    const xy_graph *g = pt->g;
    const int S = g->S, N = g->N, QS = g->q_stride;
    std::vector<int4> h(static_cast<size_t>(S) * QS * nw);
    std::vector<long long> pre(static_cast<size_t>(N) + 1), rowoff(static_cast<size_t>(N) + 1);
    std::vector<int> cut(static_cast<size_t>(nw) + 1);
    for (int s = 0; s < S; ++s) {
        const uint32_t *dg = g->h_deg.data() + static_cast<size_t>(s) * N;
        const int32_t *cp = g->h_class_ptr.data() + static_cast<size_t>(s) * QS;
        rowoff[0] = g->h_off[s];
        for (int i = 0; i < N; ++i) rowoff[i + 1] = rowoff[i] + static_cast<long long>(dg[i] & 0xffffu);
        for (int c = 0; c < QS; ++c) {
            const bool meas = c == QS - 1;
            const int cbeg = meas ? 0 : cp[c], cend = meas ? N : cp[c + 1];
            pre[0] = 0;
            for (int i = cbeg; i < cend; ++i) {
                const int deg = static_cast<int>(dg[i] & 0xffffu), nlow = static_cast<int>(dg[i] >> 16);
                pre[i - cbeg + 1] = pre[i - cbeg] + (meas ? 10 + nlow : 12 + deg);
            }
            const long long total = pre[cend - cbeg];
            int pos = 0;
            for (int k = 0; k <= nw; ++k) {
                const long long target = (total * k + nw / 2) / nw;
                while (pos < cend - cbeg && pre[pos] < target) ++pos;
                cut[k] = cbeg + pos;
            }
            cut[0] = cbeg; cut[nw] = cend;
            int4 *row = h.data() + (static_cast<size_t>(s) * QS + c) * nw;
            for (int k = 0; k < nw; ++k) {
                // the share's first chunk as the kernel will cut it (chunk_fit): the longest prefix of <= 32 sites whose
                // neighbour ids fit the staging slice -- so the ids can be staged without waiting for rec[]
                const int i0 = cut[k], w1 = cut[k + 1];
                const int nsite = std::min(32, w1 - i0);
                int msite = 0;
                while (msite < nsite && rowoff[i0 + msite + 1] - rowoff[i0] <= xy::kStageCap) ++msite;
                const int n_run = msite > 0 ? static_cast<int>(rowoff[i0 + msite] - rowoff[i0]) : 0;
                row[k] = make_int4(i0, w1, i0 < w1 ? static_cast<int>(rowoff[i0]) : 0, n_run);
            }
        }
    }
    int4 *d = nullptr;
    const int rc = dev_alloc(&d, h.size());
    if (rc != XY_OK) return rc;
    const cudaError_t e = cudaMemcpy(d, h.data(), h.size() * sizeof(int4), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(d); return fail(XY_ECUDA, std::string("share table upload: ") + cudaGetErrorString(e)); }
    pt->parts[nw] = d;
    *out = d;
    return XY_OK;
}

// CTA shape and CTAs per (sample, column block) for a launch over a group of ns samples whose largest class has nmax
// sites: one wave of resident CTAs shared by the group, at most one row per warp.  The shape is chosen per group from
// the whole sweep (all launches of a group alike): 32-warp CTAs when a warp gets at least 32 rows per sweep.
// The measuring modes (3, 5) carry the fixed-point partial sums on top of the update's state and spill at 64 registers:
// MODE 3 (over-relaxation + measurement) runs 28-warp CTAs (896 threads, 72 registers, no spills), MODE 5 (interleaved +
// measurement) 24-warp CTAs (768 threads, 80 registers; at 72 it spills ~100 bytes).  Measured on config 4: 24 instead of
// 32 warps +25 % on the interleaved cycle and +6 % on the default one; 28 instead of 24 for MODE 3 another +2 %.
struct SweepGrid { int big, gx, warps; };
SweepGrid sweep_grid(const xy_pt *pt, int ns, int nmax, int mode) {
    const int spw = 32 / pt->fast_G;
    const long long rows = static_cast<long long>(ceil_div(pt->g->N, spw)) * ns * pt->col_blocks;
    SweepGrid g;
    g.big = pt->cta_shape == 2 || (pt->cta_shape == 0 && rows >= 32ll * xy::kWarpsBig * pt->capacity_big);
    if (g.big && pt->capacity_big < ns * pt->col_blocks) g.big = 0;
    g.warps = g.big ? (mode == 3 ? 28 : mode == 5 ? 24 : xy::kWarpsBig) : xy::kWarpsSmall;
    const int cap = g.big ? pt->capacity_big : pt->sweep_capacity;
    g.gx = std::max(1, std::min(ceil_div(nmax, g.warps * spw), cap / (ns * pt->col_blocks)));
    return g;
}

xy::SweepArgs sweep_args(xy_pt *pt, int s0) {
    xy::SweepArgs a;
    a.t = tile_args(pt, 0, s0);
    a.part = nullptr;
    return a;
}

// launch attribute that keeps theta of samples s0..s1-1 resident in the persisting part of L2 while the group's
// kernels run (sample-major time blocking): every neighbour gather of the group hits this window.
// Returns 0 when the device has no persisting L2 or the option is off.
int l2_window_attr(const xy_pt *pt, int s0, int s1, cudaLaunchAttribute *attr) {
    if (!pt->l2_persist || pt->l2_persist_bytes == 0 || pt->l2_window_max == 0) return 0;
    const size_t per_sample = static_cast<size_t>(pt->g->N) * pt->R * sizeof(float);
    const size_t bytes = std::min(per_sample * static_cast<size_t>(s1 - s0), pt->l2_window_max);
    attr->id = cudaLaunchAttributeAccessPolicyWindow;
    attr->val.accessPolicyWindow.base_ptr = pt->theta + static_cast<size_t>(s0) * pt->g->N * pt->R;
    attr->val.accessPolicyWindow.num_bytes = bytes;
    attr->val.accessPolicyWindow.hitRatio = static_cast<float>(std::min(1.0, static_cast<double>(pt->l2_persist_bytes) / static_cast<double>(bytes)));
    attr->val.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    attr->val.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
    return 1;
}

// one phase (mode 0 Metropolis / 1 over-relaxation on `colour`, 2 measure) of samples s0..s1-1 as one k_phase launch
// with a programmatic-dependent-launch edge to its predecessor in the stream
int launch_phase(xy_pt *pt, int mode, int colour, int s0, int s1, bool use_counter, int sweep_offset, uint32_t sweep_fixed,
                 int accumulate /* bit 0: add to the accumulators; bit 1 (mode 3): this launch converts the sums */) {
    const xy_graph *g = pt->g;
    const int nmax = mode == 2 ? g->N : max_class_size(g, colour, s0, s1);
    if (nmax == 0 || s1 <= s0) return XY_OK;
    xy::SweepArgs a = sweep_args(pt, s0);
    a.t.colour = colour;
    a.t.sweep_fixed = sweep_fixed; a.t.sweep_offset = sweep_offset; a.t.use_counter = use_counter ? 1 : 0;
    a.t.accumulate = accumulate;
    const SweepGrid sg = sweep_grid(pt, s1 - s0, nmax, mode);
    const void *fn = (sg.warps == 24 || sg.warps == 28) ? pt->phase_fn24[mode == 5] : pt->phase_fn[sg.big][mode];
    if (pt->balance) {
        const int rc = get_partition(pt, sg.gx * sg.warps, &a.part);
        if (rc != XY_OK) return rc;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(sg.gx, s1 - s0, pt->col_blocks);
    cfg.blockDim = dim3(sg.warps * 32);
    cfg.dynamicSmemBytes = xy::sweep_smem(sg.warps);
    cfg.stream = pt->stream;
    cudaLaunchAttribute attr[2];
    int na = l2_window_attr(pt, s0, s1, &attr[0]);
    if (pt->pdl) {
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    cfg.attrs = attr; cfg.numAttrs = na;
    void *params[] = {&a};
    XY_CUDA(cudaLaunchKernelExC(&cfg, fn, params));
    pt->launches += 1;
    return XY_OK;
}

// ---- launch path with one launch per colour class, captured in CUDA graphs: k_phase for the float2 flavours,
// the any-R kernels when R has none (odd R, R = 6, 10, ...) ----
template <int MODE>
int launch_class(xy_pt *pt, int colour, int s0, int s1, bool use_counter, int sweep_offset, uint32_t sweep_fixed) {
    if (pt->fast_G) return launch_phase(pt, MODE, colour, s0, s1, use_counter, sweep_offset, sweep_fixed, 0);
    const xy_graph *g = pt->g;
    const int nmax = max_class_size(g, colour, s0, s1);
    if (nmax == 0 || s1 <= s0) return XY_OK;
    xy::TileArgs a = tile_args(pt, colour, s0);
    a.sweep_fixed = sweep_fixed; a.sweep_offset = sweep_offset; a.use_counter = use_counter ? 1 : 0;
    const long long total = static_cast<long long>(nmax) * (s1 - s0);
    // enough warps for ~3 full waves of resident warps, at most 8 sites per warp
    a.tiles_per_warp = static_cast<int>(std::min<long long>(8, std::max<long long>(1, total / (static_cast<long long>(g->n_sm) * 32 * 3))));
    const dim3 grid(ceil_div(ceil_div(nmax, a.tiles_per_warp), xy::kWarps), s1 - s0, 1);
    xy::k_update_class_generic<MODE><<<grid, xy::kBlock, 0, pt->stream>>>(a);
    XY_CUDA(cudaGetLastError());
    pt->launches += 1;
    return XY_OK;
}

int launch_measure(xy_pt *pt, int s0, int s1, bool accumulate) {
    if (pt->fast_G) return launch_phase(pt, 2, 0, s0, s1, false, 0, 0u, accumulate ? 1 : 0);
    const xy_graph *g = pt->g;
    if (s1 <= s0) return XY_OK;
    xy::TileArgs a = tile_args(pt, 0, s0);
    a.accumulate = accumulate ? 1 : 0;
    const dim3 grid(ceil_div(g->N, pt->measure_chunk), s1 - s0);
    xy::k_measure_generic<<<grid, xy::kBlock, 0, pt->stream>>>(a, pt->measure_chunk);
    XY_CUDA(cudaGetLastError());
    pt->launches += 1;
    return XY_OK;
}

xy::SwapArgs swap_args(const xy_pt *pt, const uint8_t *decisions_dev) {
    xy::SwapArgs a;
    a.E_slot = pt->E_slot; a.betaT = pt->betaT; a.beta_f = pt->beta_f; a.w_f = pt->w_f;
    a.slot_of_temp = pt->slot_of_temp; a.temp_of_slot = pt->temp_of_slot;
    a.beta_slot = pt->beta_slot; a.w_slot = pt->w_slot; a.counters = pt->counters; a.decisions = decisions_dev;
    a.attempts = pt->attempts; a.accepts = pt->accepts; a.R = pt->R;
    a.keys = pt->keys; a.sample_base = pt->sample_base;
    return a;
}

int launch_swap(xy_pt *pt, const uint8_t *decisions_dev, uint32_t d_sweep) {
    const xy::SwapArgs a = swap_args(pt, decisions_dev);
    xy::k_pt_swap<<<pt->g->S, 128, 0, pt->stream>>>(a);
    XY_CUDA(cudaGetLastError());
    xy::k_tick<<<1, 1, 0, pt->stream>>>(pt->counters, d_sweep, 1u);
    XY_CUDA(cudaGetLastError());
    pt->launches += 2;
    return XY_OK;
}

// the last non-empty colour class of samples s0..s1-1 (-1: none)
int last_colour(const xy_graph *g, int s0, int s1) {
    int last = -1;
    for (int c = 0; c < g->q_max; ++c)
        if (max_class_size(g, c, s0, s1) > 0) last = c;
    return last;
}

int sweep_group(xy_pt *pt, int mode, int s0, int s1, bool use_counter, int sweep_offset, uint32_t sweep_fixed) {
    for (int c = 0; c < pt->g->q_max; ++c) {
        const int rc = mode == 0 ? launch_class<0>(pt, c, s0, s1, use_counter, sweep_offset, sweep_fixed)
                                 : launch_class<1>(pt, c, s0, s1, false, 0, 0u);
        if (rc != XY_OK) return rc;
    }
    return XY_OK;
}

int auto_group(const xy_pt *pt) {
    const xy_graph *g = pt->g;
    int group;
    const double per_sample = static_cast<double>(g->N) * pt->R * 4.0 + static_cast<double>(g->bytes_per_sample);
    const double l2_budget = 96.0e6;  // of the 126 MB L2
    if (pt->samples_per_group > 0) group = std::min(pt->samples_per_group, g->S);
    else if (per_sample * g->S <= l2_budget) group = g->S;
    else group = std::max(1, std::min(g->S, static_cast<int>(l2_budget / per_sample)));
    if (pt->fast_G) group = std::max(1, std::min(group, pt->sweep_capacity / pt->col_blocks));   // >= 1 CTA per (sample, block)
    return group;
}

// enqueue one PT cycle on the stream; `phase` = sweep counter mod measure_every at entry
// one over-relaxation sweep of samples s0..s1-1 whose launches also produce the sweep's E, Mx, My (k_phase MODE 3);
// the launch of the last non-empty colour class converts the sums (and accumulates them when `accumulate`)
int sweep_group_fused(xy_pt *pt, int s0, int s1, bool accumulate) {
    const int last = last_colour(pt->g, s0, s1);
    if (last < 0) return launch_measure(pt, s0, s1, accumulate);
    for (int c = 0; c <= last; ++c) {
        const int rc = launch_phase(pt, 3, c, s0, s1, false, 0, 0u, (accumulate ? 1 : 0) | (c == last ? 2 : 0));
        if (rc != XY_OK) return rc;
    }
    return XY_OK;
}

// interleaved order: one sweep = for every colour class, Metropolis and then over-relaxation of each of its sites from
// one gather (k_phase MODE 4; MODE 5 also produces E, Mx, My, converted by the launch of the last non-empty colour)
int sweep_group_interleaved(xy_pt *pt, int s0, int s1, int sweep_offset, int measure /*0 none, 1 E only, 2 accumulate*/) {
    const int last = last_colour(pt->g, s0, s1);
    for (int c = 0; c <= last; ++c) {
        const int rc = launch_phase(pt, measure ? 5 : 4, c, s0, s1, true, sweep_offset, 0u,
                                    (measure == 2 ? 1 : 0) | (measure && c == last ? 2 : 0));
        if (rc != XY_OK) return rc;
    }
    if (measure && last < 0) return launch_measure(pt, s0, s1, measure == 2);
    return XY_OK;
}

int issue_cycle(xy_pt *pt, int sps, int orps, int me, int phase, int group, bool await_upload) {
    const int S = pt->g->S;
    for (int s0 = 0; s0 < S; s0 += group) {
        const int s1 = std::min(S, s0 + group);
        // xy_set_theta_async: this group's angles arrive on the copy stream; an external event-wait node orders the
        // group's first launch after its upload, so the upload of group g+1 overlaps the sweeps of group g
        if (await_upload) XY_CUDA(cudaStreamWaitEvent(pt->stream, pt->upload_ev[s0 / group], cudaEventWaitExternal));
        bool fresh = false;
        for (int k = 1; k <= sps; ++k) {
            if (pt->order == 1) {
                const bool measured = me > 0 && (phase + k) % me == 0;
                const int rc = sweep_group_interleaved(pt, s0, s1, k, measured ? 2 : (k == sps ? 1 : 0));
                if (rc != XY_OK) return rc;
                fresh = measured || k == sps;
                continue;
            }
            int rc = sweep_group(pt, 0, s0, s1, true, k, 0u);
            if (rc != XY_OK) return rc;
            const bool measured = me > 0 && (phase + k) % me == 0;
            // E is needed after this sweep: for the accumulators, or (last sweep of the cycle) for the swap round
            const bool need_e = measured || k == sps;
            const bool fuse = need_e && pt->fast_G && pt->fuse_measure && orps > 0;
            for (int o = 0; o < orps; ++o) {
                if (fuse && o == orps - 1) rc = sweep_group_fused(pt, s0, s1, measured);
                else rc = sweep_group(pt, 1, s0, s1, false, 0, 0u);
                if (rc != XY_OK) return rc;
            }
            fresh = fuse;
            if (measured && !fuse) {
                if ((rc = launch_measure(pt, s0, s1, true)) != XY_OK) return rc;
                fresh = true;
            }
        }
        if (!fresh) {
            const int rc = launch_measure(pt, s0, s1, false);
            if (rc != XY_OK) return rc;
        }
    }
    return launch_swap(pt, nullptr, static_cast<uint32_t>(sps));
}

// enqueue `sps` bare sweeps (Metropolis + orps x OR) per sample group, then advance the sweep counter
int issue_sweeps(xy_pt *pt, int sps, int orps, int group) {
    const int S = pt->g->S;
    for (int s0 = 0; s0 < S; s0 += group) {
        const int s1 = std::min(S, s0 + group);
        for (int k = 1; k <= sps; ++k) {
            if (pt->order == 1) {
                const int rc = sweep_group_interleaved(pt, s0, s1, k, 0);
                if (rc != XY_OK) return rc;
                continue;
            }
            int rc = sweep_group(pt, 0, s0, s1, true, k, 0u);
            if (rc != XY_OK) return rc;
            for (int o = 0; o < orps; ++o)
                if ((rc = sweep_group(pt, 1, s0, s1, false, 0, 0u)) != XY_OK) return rc;
        }
    }
    xy::k_tick<<<1, 1, 0, pt->stream>>>(pt->counters, static_cast<uint32_t>(sps), 0u);
    XY_CUDA(cudaGetLastError());
    pt->launches += 1;
    return XY_OK;
}

// ---- the cluster path (k_cycle): one thread-block cluster per sample runs whole cycles in one launch; its warps keep
// their rows resident in shared memory (xy_cycle.cuh) ----
// Plan: the largest cluster size C in {8, 4, 2, 1} whose per-warp pool (descriptors + neighbour ids of the rows dealt to a
// warp, maximum over warps and samples) fits a CTA's shared memory AND for which all S clusters are resident at once
// (cudaOccupancyMaxActiveClusters with the launch's real shared-memory size: cluster placement is per GPC, so fewer than
// n_sm / C clusters may fit).  If no C has room for all samples at once, the largest C that fits is used and the clusters
// run in waves (samples are independent).  Host bookkeeping only.
void cycle_plan(xy_pt *pt) {
    if (pt->cycle_planned) return;
    pt->cycle_planned = -1;
    const xy_graph *g = pt->g;
    if (!pt->fast_G || pt->col_blocks != 1 || pt->cycle_smem_max <= 0) return;
    if (g->q_max > xy::kCycleMaxQ || g->max_degree > 255) return;
    const int G = pt->fast_G, spw = 32 / G, S = g->S, N = g->N, QS = g->q_stride;
    int fallback_C = 0, fallback_k = 0, fallback_ids = 0;
    for (int C = pt->cycle_C_max; C >= 1; C /= 2) {
        const int W = xy::kCycleWarps, nw = C * W;
        std::vector<int> rows(nw), ids(nw);
        int k_cap = 0, id_cap = 0;
        for (int s = 0; s < S; ++s) {      // the ownership rule of k_cycle (xy_cycle.cuh): CTA b owns a contiguous range of every class
            std::fill(rows.begin(), rows.end(), 0);
            std::fill(ids.begin(), ids.end(), 0);
            const uint32_t *dg = g->h_deg.data() + static_cast<size_t>(s) * N;
            const int32_t *cp = g->h_class_ptr.data() + static_cast<size_t>(s) * QS;
            std::vector<int> nu0(C, 0);                                  // rows of the earlier classes per CTA
            for (int c = 0; c < g->q_max; ++c) {
                const int n_rows = (cp[c + 1] - cp[c] + spw - 1) / spw;
                for (int b = 0; b < C; ++b) {
                    const int k0 = xy::cycle_first_row(b, n_rows, C), k1 = xy::cycle_first_row(b + 1, n_rows, C);
                    for (int k = k0; k < k1; ++k) {
                        const int owner = b * W + (nu0[b] + k - k0) % W;
                        rows[owner] += 1;
                        for (int i = cp[c] + k * spw; i < std::min(cp[c] + (k + 1) * spw, cp[c + 1]); ++i)
                            ids[owner] += static_cast<int>(dg[i] & 0xffffu);
                    }
                    nu0[b] += k1 - k0;
                }
            }
            k_cap = std::max(k_cap, *std::max_element(rows.begin(), rows.end()));
            id_cap = std::max(id_cap, *std::max_element(ids.begin(), ids.end()));
        }
        k_cap = std::max(k_cap, 1);
        id_cap = std::max((id_cap + 3) / 4 * 4, 4);
        if (id_cap > 0xffff) continue;
        const size_t smem = xy::cycle_pool_bytes(G, k_cap, id_cap) * xy::kCycleWarps;
        if (smem > static_cast<size_t>(pt->cycle_smem_max)) continue;
        if (!fallback_C) { fallback_C = C; fallback_k = k_cap; fallback_ids = id_cap; }
        cudaLaunchConfig_t qc = {};
        cudaLaunchAttribute qa;
        qa.id = cudaLaunchAttributeClusterDimension;
        qa.val.clusterDim.x = C; qa.val.clusterDim.y = 1; qa.val.clusterDim.z = 1;
        qc.gridDim = dim3(C, 1, 1); qc.blockDim = dim3(xy::kCycleWarps * 32);
        qc.dynamicSmemBytes = smem;
        qc.attrs = &qa; qc.numAttrs = 1;
        int n_active = 0;
        if (cudaOccupancyMaxActiveClusters(&n_active, pt->cycle_fn[0], &qc) != cudaSuccess) { cudaGetLastError(); continue; }
        if (n_active >= S) {
            pt->cycle_C = C; pt->cycle_k_cap = k_cap; pt->cycle_id_cap = id_cap; pt->cycle_resident = 1; pt->cycle_planned = 1;
            return;
        }
    }
    if (fallback_C) {
        pt->cycle_C = fallback_C; pt->cycle_k_cap = fallback_k; pt->cycle_id_cap = fallback_ids; pt->cycle_resident = 0;
        pt->cycle_planned = 1;
    }
}

// the cluster path serves one column block (R = 2G <= 64) with at least one over-relaxation sweep per Metropolis sweep,
// samples whose rows fit the warps' resident pools, at most kCycleMaxQ colours and degrees <= 255
bool cycle_eligible(xy_pt *pt, int orps) {
    if (!(pt->fast_G && pt->col_blocks == 1 && orps >= 1 && pt->fuse_measure)) return false;
    cycle_plan(pt);
    return pt->cycle_planned == 1;
}

// automatic choice (measured): the cluster path wins while a class is a few rows per warp -- the serial
// chain of one class (barrier, one L2 round trip, the update) is then what a sweep costs -- and all samples' clusters are
// resident at once; with many rows per warp the per-launch path's 32 warps per SM and cost-balanced shares are faster.
bool use_cycle_path(xy_pt *pt, int orps) {
    if (pt->path == 1 || !cycle_eligible(pt, orps)) return false;
    if (pt->path == 2) return true;
    return pt->cycle_resident && pt->cycle_k_cap <= xy::kCycleAutoRows;
}

int launch_cycle(xy_pt *pt, int n_cycles, int sps, int orps, int me, bool do_swap) {
    const xy_graph *g = pt->g;
    if (n_cycles <= 0) return XY_OK;
    const int C = pt->cycle_C;
    xy::CycleArgs a;
    a.t = tile_args(pt, 0, 0);
    a.sw = swap_args(pt, nullptr);
    a.n_cycles = n_cycles; a.sps = sps; a.orps = orps; a.me = me; a.q_max = g->q_max; a.do_swap = do_swap ? 1 : 0;
    a.k_cap = pt->cycle_k_cap; a.id_cap = pt->cycle_id_cap;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(C, g->S, 1);
    cfg.blockDim = dim3(xy::kCycleWarps * 32);
    cfg.dynamicSmemBytes = xy::cycle_pool_bytes(pt->fast_G, a.k_cap, a.id_cap) * xy::kCycleWarps;
    cfg.stream = pt->stream;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    int na = 1;
    na += l2_window_attr(pt, 0, g->S, &attr[na]);
    cfg.attrs = attr; cfg.numAttrs = na;
    void *params[] = {&a};
    XY_CUDA(cudaLaunchKernelExC(&cfg, pt->cycle_fn[pt->order], params));
    xy::k_tick<<<1, 1, 0, pt->stream>>>(pt->counters, static_cast<uint32_t>(n_cycles) * static_cast<uint32_t>(sps),
                                        do_swap ? static_cast<uint32_t>(n_cycles) : 0u);
    XY_CUDA(cudaGetLastError());
    pt->launches += 2;
    return XY_OK;
}

// build (outside stream capture: they allocate and copy) the share tables every k_phase launch of a cycle will use
int prepare_partitions(xy_pt *pt, int group) {
    if (!pt->fast_G || !pt->balance) return XY_OK;
    const xy_graph *g = pt->g;
    for (int s0 = 0; s0 < g->S; s0 += group) {
        const int s1 = std::min(g->S, s0 + group);
        for (int c = 0; c <= g->q_max; ++c) {
            const int nmax = c == g->q_max ? g->N : max_class_size(g, c, s0, s1);
            if (nmax == 0) continue;
            const int4 *unused = nullptr;
            for (int mode : {0, 3, 5}) {      // the update shapes and the two measuring shapes
                if (c == g->q_max && mode != 0) continue;
                const SweepGrid sg = sweep_grid(pt, s1 - s0, nmax, c == g->q_max ? 2 : mode);
                const int rc = get_partition(pt, sg.gx * sg.warps, &unused);
                if (rc != XY_OK) return rc;
            }
        }
    }
    return XY_OK;
}

// capture `issue` into an executable graph stored under `key` (or fetch it from the cache)
template <typename F>
int cached_graph(xy_pt *pt, const CycleKey &key, F issue, CycleGraph **out) {
    auto it = pt->graphs.find(key);
    if (it == pt->graphs.end()) {
        if (pt->graphs.size() >= 32) {
            for (auto &kv : pt->graphs)
                if (kv.second.exec) cudaGraphExecDestroy(kv.second.exec);
            pt->graphs.clear();
        }
        cudaGraph_t graph = nullptr;
        const long long before = pt->launches;
        XY_CUDA(cudaStreamBeginCapture(pt->stream, cudaStreamCaptureModeThreadLocal));
        const int rc = issue();
        const cudaError_t e = cudaStreamEndCapture(pt->stream, &graph);
        CycleGraph cg;
        cg.launches = pt->launches - before;
        pt->launches = before;
        if (rc != XY_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (e != cudaSuccess) return fail(XY_ECUDA, std::string("cudaStreamEndCapture: ") + cudaGetErrorString(e));
        const cudaError_t e2 = cudaGraphInstantiate(&cg.exec, graph, 0);
        cudaGraphDestroy(graph);
        if (e2 != cudaSuccess) return fail(XY_ECUDA, std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e2));
        it = pt->graphs.emplace(key, cg).first;
    }
    *out = &it->second;
    return XY_OK;
}

void drop_graphs(xy_pt *pt) {
    for (auto &kv : pt->graphs)
        if (kv.second.exec) cudaGraphExecDestroy(kv.second.exec);
    pt->graphs.clear();
}

bool check_pt(const xy_pt *pt) { return pt && pt->g; }

// order the compute stream after every upload of xy_set_theta_async that is still in flight (calls other than xy_run)
int settle_upload(xy_pt *pt) {
    if (!pt->upload_armed) return XY_OK;
    pt->upload_armed = false;
    if (!pt->upload_ev.empty()) XY_CUDA(cudaStreamWaitEvent(pt->stream, pt->upload_ev.back(), 0));
    return XY_OK;
}

}  // namespace

// ====================================================================================================
extern "C" {

const char *xy_last_error(void) { return g_err.c_str(); }
int xy_abi_version(void) { return 1; }

int xy_graph_load(int S, int N, const int32_t *row_ptr, const int32_t *col_idx, const int32_t *colour,
                  void *stream, xy_graph **out) {
    if (!out) return fail(XY_EINVAL, "out is NULL");
    *out = nullptr;
    if (S < 1 || N < 1 || !row_ptr || !colour) return fail(XY_EINVAL, "need S >= 1, N >= 1, non-NULL arrays");
    try {
        // ---- validation (host) ----
        std::vector<long long> off(static_cast<size_t>(S) + 1, 0);
        int q_max = 0, max_deg = 0;
        for (int s = 0; s < S; ++s) {
            const int32_t *rp = row_ptr + static_cast<size_t>(s) * (N + 1);
            if (rp[0] != 0) return fail(XY_EGRAPH, "row_ptr[s][0] != 0 (sample " + std::to_string(s) + ")");
            for (int i = 0; i < N; ++i) {
                if (rp[i + 1] < rp[i]) return fail(XY_EGRAPH, "row_ptr not monotone (sample " + std::to_string(s) + ")");
                max_deg = std::max(max_deg, rp[i + 1] - rp[i]);
                if (rp[i + 1] - rp[i] > 0xffff) return fail(XY_EGRAPH, "degree exceeds 65535 (sample " + std::to_string(s) + ")");
            }
            off[s + 1] = off[s] + rp[N];
        }
        if (off[S] > 0 && !col_idx) return fail(XY_EINVAL, "col_idx is NULL");
        if (off[S] > 0x7fffffffll) return fail(XY_EINVAL, "total nnz exceeds int32");
        std::vector<uint64_t> fwd, rev;
        for (int s = 0; s < S; ++s) {
            const int32_t *rp = row_ptr + static_cast<size_t>(s) * (N + 1);
            const int32_t *ci = col_idx + off[s];
            const int32_t *col = colour + static_cast<size_t>(s) * N;
            const std::string where = " (sample " + std::to_string(s) + ")";
            for (int i = 0; i < N; ++i) {
                if (col[i] < 0) return fail(XY_EGRAPH, "negative colour" + where);
                if (i > 0 && col[i] < col[i - 1])
                    return fail(XY_EGRAPH, "site numbering is not colour-major (colour must be non-decreasing)" + where);
            }
            q_max = std::max(q_max, col[N - 1] + 1);
            fwd.clear(); rev.clear();
            fwd.reserve(rp[N]); rev.reserve(rp[N]);
            for (int i = 0; i < N; ++i)
                for (int e = rp[i]; e < rp[i + 1]; ++e) {
                    const int j = ci[e];
                    if (j < 0 || j >= N) return fail(XY_EGRAPH, "neighbour id out of range" + where);
                    if (j == i) return fail(XY_EGRAPH, "self-loop" + where);
                    if (col[j] == col[i]) return fail(XY_EGRAPH, "monochromatic edge: colouring is not proper" + where);
                    fwd.push_back((static_cast<uint64_t>(i) << 32) | static_cast<uint32_t>(j));
                    rev.push_back((static_cast<uint64_t>(j) << 32) | static_cast<uint32_t>(i));
                }
            std::sort(fwd.begin(), fwd.end());
            std::sort(rev.begin(), rev.end());
            if (std::adjacent_find(fwd.begin(), fwd.end()) != fwd.end()) return fail(XY_EGRAPH, "duplicate edge" + where);
            if (fwd != rev) return fail(XY_EGRAPH, "adjacency is not symmetric" + where);
        }
        // ---- device copies ----
        int n_dev = 0;
        if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1)
            return fail(XY_ECUDA, "no CUDA device: this library has no CPU fallback");
        xy_graph *g = new xy_graph();
        if (cudaGetDevice(&g->device) != cudaSuccess ||
            cudaDeviceGetAttribute(&g->n_sm, cudaDevAttrMultiProcessorCount, g->device) != cudaSuccess || g->n_sm < 1) {
            delete g;
            return fail(XY_ECUDA, "cannot query the current CUDA device");
        }
        g->S = S; g->N = N; g->q_max = q_max; g->q_stride = q_max + 1; g->max_degree = max_deg;
        g->nnz_total = off[S];
        g->stream = static_cast<cudaStream_t>(stream);
        g->bytes_per_sample = static_cast<size_t>(off[S] / S) * 4 + static_cast<size_t>(N) * 8;
        std::vector<int2> h_rec(static_cast<size_t>(S) * N);
        std::vector<int32_t> h_col(static_cast<size_t>(off[S]));   // neighbour lists, ascending per site
        g->h_class_ptr.assign(static_cast<size_t>(S) * g->q_stride, 0);
        g->h_deg.assign(static_cast<size_t>(S) * N, 0u);
        g->h_off = off;
        for (int s = 0; s < S; ++s) {
            const int32_t *rp = row_ptr + static_cast<size_t>(s) * (N + 1);
            const int32_t *col = colour + static_cast<size_t>(s) * N;
            int32_t *cp = g->h_class_ptr.data() + static_cast<size_t>(s) * g->q_stride;
            for (int i = 0; i < N; ++i) {
                int32_t *dst = h_col.data() + off[s] + rp[i];
                const int deg = rp[i + 1] - rp[i];
                std::copy(col_idx + off[s] + rp[i], col_idx + off[s] + rp[i + 1], dst);
                std::sort(dst, dst + deg);
                const int n_lower = static_cast<int>(std::lower_bound(dst, dst + deg, i) - dst);
                h_rec[static_cast<size_t>(s) * N + i] = make_int2(static_cast<int>(off[s] + rp[i]), deg | (n_lower << 16));
                g->h_deg[static_cast<size_t>(s) * N + i] = static_cast<uint32_t>(deg | (n_lower << 16));
                cp[col[i] + 1]++;
            }
            for (int c = 0; c < q_max; ++c) cp[c + 1] += cp[c];
        }
        int rc;
        if ((rc = dev_alloc(&g->rec, h_rec.size())) != XY_OK || (rc = dev_alloc(&g->col_idx, off[S])) != XY_OK ||
            (rc = dev_alloc(&g->class_ptr, g->h_class_ptr.size())) != XY_OK) {
            xy_graph_free(g);
            return rc;
        }
        cudaError_t e = cudaMemcpyAsync(g->rec, h_rec.data(), h_rec.size() * sizeof(int2), cudaMemcpyHostToDevice, g->stream);
        if (e == cudaSuccess && off[S] > 0)
            e = cudaMemcpyAsync(g->col_idx, h_col.data(), off[S] * sizeof(int32_t), cudaMemcpyHostToDevice, g->stream);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(g->class_ptr, g->h_class_ptr.data(), g->h_class_ptr.size() * sizeof(int32_t),
                                cudaMemcpyHostToDevice, g->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(g->stream);
        if (e != cudaSuccess) {
            xy_graph_free(g);
            return fail(XY_ECUDA, std::string("graph upload: ") + cudaGetErrorString(e));
        }
        *out = g;
        return XY_OK;
    } catch (const std::bad_alloc &) {
        return fail(XY_ENOMEM, "host allocation failed");
    }
}

int xy_graph_free(xy_graph *g) {
    if (!g) return XY_OK;
    DeviceGuard guard(g->device);
    cudaFree(g->rec); cudaFree(g->col_idx); cudaFree(g->class_ptr);
    cudaFree(g->coords); cudaFree(g->tab1); cudaFree(g->tab2);
    delete g;
    return XY_OK;
}

int xy_graph_set_coords(xy_graph *g, int Lx, int Ly, const int32_t *x, const int32_t *y) {
    if (!g || !x || !y) return fail(XY_EINVAL, "graph or coordinate array is NULL");
    DeviceGuard guard(g->device);
    if (Lx < 1 || Ly < 1 || Lx > 65535 || Ly > 65535) return fail(XY_EINVAL, "need 1 <= Lx, Ly <= 65535");
    const size_t n = static_cast<size_t>(g->S) * g->N;
    try {
        std::vector<uint32_t> h(n);
        for (size_t i = 0; i < n; ++i) {
            if (x[i] < 0 || x[i] >= Lx || y[i] < 0 || y[i] >= Ly) return fail(XY_EINVAL, "site coordinate out of range");
            h[i] = static_cast<uint32_t>(x[i]) | (static_cast<uint32_t>(y[i]) << 16);
        }
        std::vector<float2> t1(Lx), t2(Ly);
        const double two_pi = 6.283185307179586476925286766559;
        for (int k = 0; k < Lx; ++k) t1[k] = make_float2(static_cast<float>(std::cos(two_pi * k / Lx)), static_cast<float>(std::sin(two_pi * k / Lx)));
        for (int k = 0; k < Ly; ++k) t2[k] = make_float2(static_cast<float>(std::cos(two_pi * k / Ly)), static_cast<float>(std::sin(two_pi * k / Ly)));
        cudaFree(g->coords); cudaFree(g->tab1); cudaFree(g->tab2);
        g->coords = nullptr; g->tab1 = g->tab2 = nullptr; g->Lx = g->Ly = 0;
        int rc;
        if ((rc = dev_alloc(&g->coords, n)) != XY_OK || (rc = dev_alloc(&g->tab1, Lx)) != XY_OK ||
            (rc = dev_alloc(&g->tab2, Ly)) != XY_OK)
            return rc;
        XY_CUDA(cudaMemcpy(g->coords, h.data(), n * sizeof(uint32_t), cudaMemcpyHostToDevice));
        XY_CUDA(cudaMemcpy(g->tab1, t1.data(), Lx * sizeof(float2), cudaMemcpyHostToDevice));
        XY_CUDA(cudaMemcpy(g->tab2, t2.data(), Ly * sizeof(float2), cudaMemcpyHostToDevice));
        g->Lx = Lx; g->Ly = Ly;
    } catch (const std::bad_alloc &) {
        return fail(XY_ENOMEM, "host allocation failed");
    }
    return XY_OK;
}

int xy_random_walk(const xy_graph *g, int n_walkers, const int32_t *start, int n_steps, uint64_t seed, uint32_t sample_base,
                   void *stream, int64_t *hist_host) {
    if (!g || !start || !hist_host) return fail(XY_EINVAL, "graph, start or hist is NULL");
    DeviceGuard guard(g->device);
    if (n_walkers < 1 || n_steps < 0 || n_steps > 12000) return fail(XY_EINVAL, "need n_walkers >= 1, 0 <= n_steps <= 12000");
    if (static_cast<uint64_t>(sample_base) + g->S > 65536u) return fail(XY_EINVAL, "sample_base + S must be <= 65536");
    const size_t nw = static_cast<size_t>(g->S) * n_walkers, nh = static_cast<size_t>(g->S) * (n_steps + 1);
    for (size_t i = 0; i < nw; ++i)
        if (start[i] < 0 || start[i] >= g->N) return fail(XY_EINVAL, "start site out of range");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int32_t *d_start = nullptr;
    unsigned long long *d_hist = nullptr;
    int rc;
    if ((rc = dev_alloc(&d_start, nw)) != XY_OK) return rc;
    if ((rc = dev_alloc(&d_hist, nh)) != XY_OK) { cudaFree(d_start); return rc; }
    xy::WalkArgs a;
    a.rec = g->rec; a.col_idx = g->col_idx; a.start = d_start; a.hist = d_hist;
    a.N = g->N; a.n_walkers = n_walkers; a.n_steps = n_steps; a.sample_base = sample_base;
    a.keys = xy::philox_key_schedule(static_cast<uint32_t>(seed), static_cast<uint32_t>(seed >> 32));
    cudaEvent_t k0 = nullptr, k1 = nullptr;
    g_walk_kernel_us = -1.0;
    cudaError_t e = cudaMemcpyAsync(d_start, start, nw * sizeof(int32_t), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_hist, 0, nh * sizeof(unsigned long long), st);
    if (e == cudaSuccess) e = cudaEventCreate(&k0);
    if (e == cudaSuccess) e = cudaEventCreate(&k1);
    if (e == cudaSuccess) {
        const dim3 grid(ceil_div(n_walkers, xy::kBlock), g->S);
        cudaEventRecord(k0, st);
        xy::k_random_walk<<<grid, xy::kBlock, (n_steps + 1) * sizeof(unsigned int), st>>>(a);
        e = cudaGetLastError();
        cudaEventRecord(k1, st);
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(hist_host, d_hist, nh * sizeof(int64_t), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    float k_ms = 0.f;
    if (e == cudaSuccess && cudaEventElapsedTime(&k_ms, k0, k1) == cudaSuccess) g_walk_kernel_us = 1e3 * k_ms;
    if (k0) cudaEventDestroy(k0);
    if (k1) cudaEventDestroy(k1);
    cudaFree(d_start); cudaFree(d_hist);
    if (e != cudaSuccess) return fail(XY_ECUDA, std::string("xy_random_walk: ") + cudaGetErrorString(e));
    return XY_OK;
}

// ---- xy_random_walk_static: the walk without any allocation (include/xy_b200.h) ----
// scratch of the no-allocation entry point: the histogram words the kernel's atomics add to, plus one word that counts
// invalid start sites.  A host-side stand-in in host code: its device address comes from cudaGetSymbolAddress.
static __device__ __align__(256) unsigned long long g_walk_scratch[XY_WALK_STATIC_ENTRIES + 32];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_walk_mutex;
unsigned long long *g_walk_scratch_dev[kMaxDevices] = {};      // per device: the array's address there (set up once)

__global__ void k_walk_check_starts(const int32_t *start, size_t n, int N, unsigned long long *bad) {
    for (size_t i = blockIdx.x * static_cast<size_t>(blockDim.x) + threadIdx.x; i < n; i += static_cast<size_t>(gridDim.x) * blockDim.x)
        if (start[i] < 0 || start[i] >= N) atomicAdd(bad, 1ull);
}
}  // namespace

int xy_random_walk_static(const xy_graph *g, int n_walkers, const int32_t *start_dev, int n_steps, uint64_t seed,
                          uint32_t sample_base, void *stream, int64_t *hist_dev) {
    if (!g || !start_dev || !hist_dev) return fail(XY_EINVAL, "graph, start_dev or hist_dev is NULL");
    DeviceGuard guard(g->device);
    if (n_walkers < 1 || n_steps < 0 || n_steps > 12000) return fail(XY_EINVAL, "need n_walkers >= 1, 0 <= n_steps <= 12000");
    if (static_cast<uint64_t>(sample_base) + g->S > 65536u) return fail(XY_EINVAL, "sample_base + S must be <= 65536");
    const size_t nw = static_cast<size_t>(g->S) * n_walkers, nh = static_cast<size_t>(g->S) * (n_steps + 1);
    if (nh > static_cast<size_t>(XY_WALK_STATIC_ENTRIES))
        return fail(XY_EINVAL, "xy_random_walk_static: S * (n_steps + 1) = " + std::to_string(nh) + " exceeds the static scratch of " +
                                   std::to_string(XY_WALK_STATIC_ENTRIES) + " words; use xy_random_walk");
    if (g->device < 0 || g->device >= kMaxDevices) return fail(XY_EINVAL, "device index beyond 63");
    unsigned long long *scratch = nullptr;
    {   // set-up, once per device, with that device current (DeviceGuard above)
        std::lock_guard<std::mutex> lock(g_walk_mutex);
        if (!g_walk_scratch_dev[g->device]) {
            void *p = nullptr;
            const cudaError_t es = cudaGetSymbolAddress(&p, g_walk_scratch);
            if (es != cudaSuccess || !p) return fail(XY_ECUDA, std::string("cudaGetSymbolAddress(g_walk_scratch): ") + cudaGetErrorString(es));
            g_walk_scratch_dev[g->device] = static_cast<unsigned long long *>(p);
        }
        scratch = g_walk_scratch_dev[g->device];
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    unsigned long long *bad = scratch + XY_WALK_STATIC_ENTRIES;
    // the array keeps the last call's contents: clear the words this call uses (and the error word)
    XY_CUDA(cudaMemsetAsync(scratch, 0, nh * sizeof(unsigned long long), st));
    XY_CUDA(cudaMemsetAsync(bad, 0, sizeof(unsigned long long), st));
    k_walk_check_starts<<<std::max(1, std::min(g->n_sm * 4, ceil_div(static_cast<long long>(nw), 256))), 256, 0, st>>>(start_dev, nw, g->N, bad);
    XY_CUDA(cudaGetLastError());
    unsigned long long n_bad = 0;
    XY_CUDA(cudaMemcpyAsync(&n_bad, bad, sizeof(n_bad), cudaMemcpyDeviceToHost, st));
    XY_CUDA(cudaStreamSynchronize(st));
    if (n_bad) return fail(XY_EINVAL, "start site out of range");
    xy::WalkArgs a;
    a.rec = g->rec; a.col_idx = g->col_idx; a.start = start_dev; a.hist = scratch;
    a.N = g->N; a.n_walkers = n_walkers; a.n_steps = n_steps; a.sample_base = sample_base;
    a.keys = xy::philox_key_schedule(static_cast<uint32_t>(seed), static_cast<uint32_t>(seed >> 32));
    const dim3 grid(ceil_div(n_walkers, xy::kBlock), g->S);
    xy::k_random_walk<<<grid, xy::kBlock, (n_steps + 1) * sizeof(unsigned int), st>>>(a);
    XY_CUDA(cudaGetLastError());
    XY_CUDA(cudaMemcpyAsync(hist_dev, scratch, nh * sizeof(int64_t), cudaMemcpyDeviceToDevice, st));
    XY_CUDA(cudaStreamSynchronize(st));
    return XY_OK;
}

int xy_random_walk_kernel_us(double *us_out) {
    if (!us_out) return fail(XY_EINVAL, "NULL output");
    if (g_walk_kernel_us < 0.0) return fail(XY_ESTATE, "no successful xy_random_walk call on this thread yet");
    *us_out = g_walk_kernel_us;
    return XY_OK;
}

int xy_graph_info(const xy_graph *g, int *S, int *N, int64_t *nnz_total, int *q_max, int *max_degree) {
    if (!g) return fail(XY_EINVAL, "graph is NULL");
    if (S) *S = g->S;
    if (N) *N = g->N;
    if (nnz_total) *nnz_total = g->nnz_total;
    if (q_max) *q_max = g->q_max;
    if (max_degree) *max_degree = g->max_degree;
    return XY_OK;
}

int xy_pt_create(const xy_graph *g, int R, const double *T, const double *width, uint64_t seed, uint32_t sample_base,
                 float *theta_dev, void *stream, xy_pt **out) {
    if (!out) return fail(XY_EINVAL, "out is NULL");
    *out = nullptr;
    if (!g || !T) return fail(XY_EINVAL, "graph or T is NULL");
    DeviceGuard guard(g->device);
    if (R < 1 || R > 1024) return fail(XY_EINVAL, "need 1 <= R <= 1024");
    if (static_cast<uint64_t>(sample_base) + g->S > 65536u) return fail(XY_EINVAL, "sample_base + S must be <= 65536");
    for (int k = 0; k < R; ++k) {
        if (!(T[k] > 0.0)) return fail(XY_EINVAL, "temperatures must be > 0");
        if (k > 0 && !(T[k] >= T[k - 1])) return fail(XY_EINVAL, "temperatures must be ascending");
        // R5 wraps a proposal once by +-2 pi: |delta| <= width / 2 must not exceed 2 pi
        if (width && !(width[k] >= 0.0 && width[k] <= 4.0 * 3.14159265358979323846))
            return fail(XY_EINVAL, "proposal width must lie in [0, 4 pi]");
    }
    if (theta_dev && (reinterpret_cast<uintptr_t>(theta_dev) & 7u)) return fail(XY_EINVAL, "theta_dev must be 8-byte aligned");
    xy_pt *pt = nullptr;
    try {
        pt = new xy_pt();
    } catch (const std::bad_alloc &) {
        return fail(XY_ENOMEM, "host allocation failed");
    }
    pt->g = g; pt->R = R;
    pt->key0 = static_cast<uint32_t>(seed); pt->key1 = static_cast<uint32_t>(seed >> 32);
    pt->sample_base = sample_base;
    pt->stream = static_cast<cudaStream_t>(stream);
    if (!pt->stream) {  // CUDA graphs cannot be captured on the legacy default stream
        const cudaError_t es = cudaStreamCreateWithFlags(&pt->stream, cudaStreamNonBlocking);
        if (es != cudaSuccess) {
            delete pt;
            return fail(XY_ECUDA, std::string("cudaStreamCreate: ") + cudaGetErrorString(es));
        }
        pt->owns_stream = true;
    }
    const int S = g->S, N = g->N;
    // kernel flavour: float2 path when R = 2G with G a power of two <= 32, or R a multiple of 64
    pt->fast_G = 0; pt->col_blocks = 1;
    if (R % 64 == 0) { pt->fast_G = 32; pt->col_blocks = R / 64; }
    else if (R % 2 == 0 && R / 2 <= 32 && ((R / 2) & (R / 2 - 1)) == 0) pt->fast_G = R / 2;
    if (static_cast<long long>(N) * ((R + 1) / 2) > 0x7fffffffll) {
        if (pt->owns_stream) cudaStreamDestroy(pt->stream);
        delete pt;
        return fail(XY_EINVAL, "N * R / 2 must fit in int32 (offsets inside a sample are 32-bit)");
    }
    pt->keys = xy::philox_key_schedule(pt->key0, pt->key1);
    pt->measure_chunk = std::max(256, ((N + 127) / 128 + 7) / 8 * 8);   // legacy measure partition: a function of N only
    if (pt->fast_G) {
        cudaError_t eo = cudaSuccess;
        auto prepare = [&](const void *fn, int warps) {      // opt in to the kernel's dynamic shared memory
            if (eo == cudaSuccess)
                eo = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(xy::sweep_smem(warps)));
            if (eo == cudaSuccess)
                eo = cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, static_cast<int>(cudaSharedmemCarveoutMaxShared));
        };
        for (int m = 0; m < 6; ++m) {
            pt->phase_fn[0][m] = xy::phase_function(xy::kWarpsSmall, pt->fast_G, pt->col_blocks == 1, m);
            pt->phase_fn[1][m] = xy::phase_function(xy::kWarpsBig, pt->fast_G, pt->col_blocks == 1, m);
            prepare(pt->phase_fn[0][m], xy::kWarpsSmall);
            prepare(pt->phase_fn[1][m], xy::kWarpsBig);
        }
        // 32 resident warps x 5.5 KB of shared memory per SM in either CTA shape (carve-out set above)
        pt->phase_fn24[0] = xy::phase_function(28, pt->fast_G, pt->col_blocks == 1, 3);
        pt->phase_fn24[1] = xy::phase_function(24, pt->fast_G, pt->col_blocks == 1, 5);
        prepare(pt->phase_fn24[0], 28);
        prepare(pt->phase_fn24[1], 24);
        int per_sm = 0, per_sm_big = 0;
        const int n_sm = g->n_sm, dev = g->device;
        if (eo == cudaSuccess)
            eo = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pt->phase_fn[0][0], xy::kWarpsSmall * 32,
                                                               xy::sweep_smem(xy::kWarpsSmall));
        if (eo == cudaSuccess)
            eo = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_big, pt->phase_fn[1][0], xy::kWarpsBig * 32,
                                                               xy::sweep_smem(xy::kWarpsBig));
        if (eo != cudaSuccess || per_sm < 1) {
            if (pt->owns_stream) cudaStreamDestroy(pt->stream);
            delete pt;
            return fail(XY_ECUDA, std::string("k_phase attributes / occupancy query: ") + cudaGetErrorString(eo));
        }
        pt->sweep_capacity = per_sm * n_sm;
        pt->capacity_big = std::max(1, per_sm_big) * n_sm;
        // the cluster path (k_cycle): one column block only; opt in to all the shared memory a CTA may have (the plan made at
        // the first use sizes the launch)
        if (pt->col_blocks == 1) {
            pt->cycle_fn[0] = xy::cycle_function(0, pt->fast_G);
            pt->cycle_fn[1] = xy::cycle_function(1, pt->fast_G);
            int optin = 0;
            cudaError_t ec = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
            int dyn_max = 0;
            for (int o = 0; o < 2 && ec == cudaSuccess; ++o) {
                cudaFuncAttributes fa;
                ec = cudaFuncGetAttributes(&fa, pt->cycle_fn[o]);
                if (ec != cudaSuccess) break;
                const int room = optin - static_cast<int>(fa.sharedSizeBytes);
                dyn_max = o == 0 ? room : std::min(dyn_max, room);
                ec = cudaFuncSetAttribute(pt->cycle_fn[o], cudaFuncAttributeMaxDynamicSharedMemorySize, room);
                if (ec == cudaSuccess && cudaFuncSetAttribute(pt->cycle_fn[o], cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
                    cudaGetLastError();
                    pt->cycle_C_max = 8;
                } else if (o == 0) {
                    pt->cycle_C_max = 16;
                }
            }
            pt->cycle_smem_max = ec == cudaSuccess ? dyn_max : 0;
            cudaGetLastError();
        }
        // persisting L2 carve-out for the access-policy windows of the sample groups; xy_pt_destroy puts the limit back
        int max_persist = 0, max_window = 0;
        if (cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&max_window, cudaDevAttrMaxAccessPolicyWindowSize, dev) == cudaSuccess && max_persist > 0 &&
            max_window > 0 && l2_carveout_acquire(dev, static_cast<size_t>(max_persist))) {
            pt->l2_persist_bytes = static_cast<size_t>(max_persist);
            pt->l2_window_max = static_cast<size_t>(max_window);
            pt->l2_limit_set = true;
        }
        cudaGetLastError();
    }

    const size_t SR = static_cast<size_t>(S) * R;
    int rc = XY_OK;
    auto A = [&](int r) { if (rc == XY_OK) rc = r; };
    if (theta_dev) pt->theta = theta_dev;
    else { A(dev_alloc(&pt->theta, SR * N)); pt->owns_theta = true; }
    A(dev_alloc(&pt->beta_slot, SR)); A(dev_alloc(&pt->w_slot, SR));
    A(dev_alloc(&pt->beta_f, R)); A(dev_alloc(&pt->w_f, R)); A(dev_alloc(&pt->betaT, R));
    A(dev_alloc(&pt->temp_of_slot, SR)); A(dev_alloc(&pt->slot_of_temp, SR));
    A(dev_alloc(&pt->counters, 2));
    A(dev_alloc(&pt->E_slot, SR)); A(dev_alloc(&pt->M_slot, SR * 2));
    A(dev_alloc(&pt->fx, SR * 3 * 2)); A(dev_alloc(&pt->ticket, S)); A(dev_alloc(&pt->acc, SR * XY_NACC));
    A(dev_alloc(&pt->attempts, SR)); A(dev_alloc(&pt->accepts, SR)); A(dev_alloc(&pt->decisions, SR));
    A(dev_alloc(&pt->G_slot, SR * 2)); A(dev_alloc(&pt->acc_k, SR * 3)); A(dev_alloc(&pt->fk, SR * 8));

    if (rc != XY_OK) { xy_pt_destroy(pt); return rc; }
    std::vector<float> hb(R), hw(R);
    std::vector<double> hbT(R);
    std::vector<int32_t> lab(SR);
    for (int k = 0; k < R; ++k) {
        hbT[k] = 1.0 / T[k];
        hb[k] = static_cast<float>(1.0 / T[k]);
        const double half = 0.5 * T[k];
        hw[k] = static_cast<float>(width ? width[k] : 6.283185307179586476925286766559 * (half < 1.0 ? half : 1.0));
    }
    for (size_t i = 0; i < SR; ++i) lab[i] = static_cast<int32_t>(i % R);
    cudaError_t e = cudaMemcpyAsync(pt->beta_f, hb.data(), R * sizeof(float), cudaMemcpyHostToDevice, pt->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(pt->w_f, hw.data(), R * sizeof(float), cudaMemcpyHostToDevice, pt->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(pt->betaT, hbT.data(), R * sizeof(double), cudaMemcpyHostToDevice, pt->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(pt->temp_of_slot, lab.data(), SR * sizeof(int32_t), cudaMemcpyHostToDevice, pt->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(pt->counters, 0, 2 * sizeof(uint32_t), pt->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(pt->acc, 0, SR * XY_NACC * sizeof(double), pt->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(pt->attempts, 0, SR * sizeof(long long), pt->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(pt->accepts, 0, SR * sizeof(long long), pt->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(pt->E_slot, 0, SR * sizeof(double), pt->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(pt->fx, 0, SR * 3 * 2 * sizeof(long long), pt->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(pt->fk, 0, SR * 8 * sizeof(long long), pt->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(pt->acc_k, 0, SR * 3 * sizeof(double), pt->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(pt->G_slot, 0, SR * 2 * sizeof(double), pt->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(pt->ticket, 0, S * sizeof(unsigned int), pt->stream);
    if (e == cudaSuccess) {
        xy::k_refresh_slot_params<<<ceil_div(SR, 128), 128, 0, pt->stream>>>(pt->temp_of_slot, pt->slot_of_temp, pt->beta_f,
                                                                            pt->w_f, pt->beta_slot, pt->w_slot, S, R);
        xy::k_init_theta<<<g->n_sm * 8, 256, 0, pt->stream>>>(pt->theta, S, N, R, pt->keys, pt->sample_base);
        pt->launches += 2;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(pt->stream);
    if (e != cudaSuccess) {
        xy_pt_destroy(pt);
        return fail(XY_ECUDA, std::string("xy_pt_create: ") + cudaGetErrorString(e));
    }
    *out = pt;
    return XY_OK;
}

int xy_pt_destroy(xy_pt *pt) {
    if (!pt) return XY_OK;
    DeviceGuard guard(pt->g ? pt->g->device : -1);
    cudaStreamSynchronize(pt->stream);
    drop_graphs(pt);
    if (pt->owns_theta) cudaFree(pt->theta);
    cudaFree(pt->beta_slot); cudaFree(pt->w_slot); cudaFree(pt->beta_f); cudaFree(pt->w_f); cudaFree(pt->betaT);
    cudaFree(pt->temp_of_slot); cudaFree(pt->slot_of_temp); cudaFree(pt->counters);
    cudaFree(pt->E_slot); cudaFree(pt->M_slot); cudaFree(pt->fx); cudaFree(pt->ticket); cudaFree(pt->acc);
    cudaFree(pt->attempts); cudaFree(pt->accepts); cudaFree(pt->decisions);
    cudaFree(pt->G_slot); cudaFree(pt->acc_k); cudaFree(pt->fk);
    for (auto &kv : pt->parts) cudaFree(kv.second);
    if (pt->l2_limit_set) l2_carveout_release(pt->g->device);      // the last ensemble gives the carve-out back
    for (cudaEvent_t ev : pt->upload_ev) cudaEventDestroy(ev);
    if (pt->compute_done) cudaEventDestroy(pt->compute_done);
    if (pt->copy_stream) { cudaStreamSynchronize(pt->copy_stream); cudaStreamDestroy(pt->copy_stream); }
    if (pt->owns_stream) cudaStreamDestroy(pt->stream);
    delete pt;
    return XY_OK;
}

int xy_sweep(xy_pt *pt, int n_sweeps) {
    if (!check_pt(pt) || n_sweeps < 0) return fail(XY_EINVAL, "bad handle or n_sweeps < 0");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    for (int n = 0; n < n_sweeps; ++n) {
        const int rc = sweep_group(pt, 0, 0, pt->g->S, true, 1, 0u);
        if (rc != XY_OK) return rc;
        xy::k_tick<<<1, 1, 0, pt->stream>>>(pt->counters, 1u, 0u);
        XY_CUDA(cudaGetLastError());
        pt->launches += 1;
        pt->sweep += 1;
    }
    if (n_sweeps > 0) pt->e_fresh = false;
    return XY_OK;
}

int xy_sweep_acceptance(xy_pt *pt, double *acc_host) {
    if (!check_pt(pt) || !acc_host) return fail(XY_EINVAL, "bad handle or NULL output");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    const int S = pt->g->S, N = pt->g->N, R = pt->R;
    const size_t n = static_cast<size_t>(S) * N * R, SR = static_cast<size_t>(S) * R;
    float *before = nullptr;
    unsigned long long *count = nullptr;
    int rc;
    if ((rc = dev_alloc(&before, n)) != XY_OK) return rc;
    if ((rc = dev_alloc(&count, SR)) != XY_OK) { cudaFree(before); return rc; }
    cudaError_t e = cudaMemcpyAsync(before, pt->theta, n * sizeof(float), cudaMemcpyDeviceToDevice, pt->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(count, 0, SR * sizeof(unsigned long long), pt->stream);
    rc = e == cudaSuccess ? xy_sweep(pt, 1) : fail(XY_ECUDA, std::string("xy_sweep_acceptance: ") + cudaGetErrorString(e));
    if (rc == XY_OK) {
        const int spb = std::max(1, ceil_div(N, std::max(1, pt->g->n_sm * 8 / S)));
        xy::k_count_changed<<<dim3(ceil_div(N, spb), S), xy::kBlock, 0, pt->stream>>>(before, pt->theta, count, N, R, spb);
        pt->launches += 1;
        try {
            std::vector<unsigned long long> h(SR);
            std::vector<int32_t> tos(SR);
            e = cudaGetLastError();
            if (e == cudaSuccess) e = cudaMemcpyAsync(h.data(), count, SR * sizeof(unsigned long long), cudaMemcpyDeviceToHost, pt->stream);
            if (e == cudaSuccess) e = cudaMemcpyAsync(tos.data(), pt->temp_of_slot, SR * sizeof(int32_t), cudaMemcpyDeviceToHost, pt->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(pt->stream);
            if (e != cudaSuccess) rc = fail(XY_ECUDA, std::string("xy_sweep_acceptance: ") + cudaGetErrorString(e));
            else
                for (int s = 0; s < S; ++s)
                    for (int r = 0; r < R; ++r)
                        acc_host[static_cast<size_t>(s) * R + tos[static_cast<size_t>(s) * R + r]] =
                            static_cast<double>(h[static_cast<size_t>(s) * R + r]) / N;
        } catch (const std::bad_alloc &) {
            rc = fail(XY_ENOMEM, "host allocation failed");
        }
    }
    cudaStreamSynchronize(pt->stream);
    cudaFree(before); cudaFree(count);
    return rc;
}

int xy_overrelax(xy_pt *pt, int n_sweeps) {
    if (!check_pt(pt) || n_sweeps < 0) return fail(XY_EINVAL, "bad handle or n_sweeps < 0");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    for (int n = 0; n < n_sweeps; ++n) {
        const int rc = sweep_group(pt, 1, 0, pt->g->S, false, 0, 0u);
        if (rc != XY_OK) return rc;
    }
    if (n_sweeps > 0) pt->e_fresh = false;
    return XY_OK;
}

int xy_metropolis_colour(xy_pt *pt, int colour, uint32_t sweep) {
    if (!check_pt(pt) || colour < 0 || colour >= pt->g->q_max) return fail(XY_EINVAL, "bad handle or colour");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    pt->e_fresh = false;
    const int group = auto_group(pt);
    for (int s0 = 0; s0 < pt->g->S; s0 += group) {
        const int rc = launch_class<0>(pt, colour, s0, std::min(pt->g->S, s0 + group), false, 0, sweep);
        if (rc != XY_OK) return rc;
    }
    return XY_OK;
}

int xy_metor_colour(xy_pt *pt, int colour, uint32_t sweep) {
    if (!check_pt(pt) || colour < 0 || colour >= pt->g->q_max) return fail(XY_EINVAL, "bad handle or colour");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    if (!pt->fast_G) return fail(XY_ESTATE, "the interleaved order needs a float2 kernel flavour (R = 2 * 2^k <= 64 or R % 64 == 0)");
    pt->e_fresh = false;
    const int group = auto_group(pt);
    for (int s0 = 0; s0 < pt->g->S; s0 += group) {
        const int rc = launch_phase(pt, 4, colour, s0, std::min(pt->g->S, s0 + group), false, 0, sweep, 0);
        if (rc != XY_OK) return rc;
    }
    return XY_OK;
}

int xy_set_order(xy_pt *pt, int order) {
    if (!check_pt(pt) || order < 0 || order > 1) return fail(XY_EINVAL, "bad handle or order not in {0, 1}");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    if (order == 1 && !pt->fast_G)
        return fail(XY_ESTATE, "the interleaved order needs a float2 kernel flavour (R = 2 * 2^k <= 64 or R % 64 == 0)");
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    pt->order = order;
    drop_graphs(pt);
    return XY_OK;
}

int xy_overrelax_colour(xy_pt *pt, int colour) {
    if (!check_pt(pt) || colour < 0 || colour >= pt->g->q_max) return fail(XY_EINVAL, "bad handle or colour");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    pt->e_fresh = false;
    const int group = auto_group(pt);
    for (int s0 = 0; s0 < pt->g->S; s0 += group) {
        const int rc = launch_class<1>(pt, colour, s0, std::min(pt->g->S, s0 + group), false, 0, 0u);
        if (rc != XY_OK) return rc;
    }
    return XY_OK;
}

int xy_pt_swap(xy_pt *pt) {
    if (!check_pt(pt)) return fail(XY_EINVAL, "bad handle");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    if (!pt->e_fresh) {
        const int rc = launch_measure(pt, 0, pt->g->S, false);
        if (rc != XY_OK) return rc;
        pt->e_fresh = true;
    }
    const int rc = launch_swap(pt, nullptr, 0u);
    if (rc == XY_OK) pt->round += 1;
    return rc;
}

int xy_swap_with_decisions(xy_pt *pt, const uint8_t *accept_host) {
    if (!check_pt(pt) || !accept_host) return fail(XY_EINVAL, "bad handle or NULL decisions");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    const size_t SR = static_cast<size_t>(pt->g->S) * pt->R;
    XY_CUDA(cudaMemcpyAsync(pt->decisions, accept_host, SR, cudaMemcpyHostToDevice, pt->stream));
    XY_CUDA(cudaStreamSynchronize(pt->stream));  // accept_host is borrowed for the call only
    const int rc = launch_swap(pt, pt->decisions, 0u);
    if (rc == XY_OK) pt->round += 1;
    return rc;
}

int xy_measure(xy_pt *pt, double *out_host) {
    if (!check_pt(pt)) return fail(XY_EINVAL, "bad handle");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    const int S = pt->g->S, R = pt->R;
    const int rc = launch_measure(pt, 0, S, true);
    if (rc != XY_OK) return rc;
    pt->e_fresh = true;
    if (out_host) {
        const size_t SR = static_cast<size_t>(S) * R;
        try {
            std::vector<double> E(SR), M(SR * 2);
            std::vector<int32_t> tos(SR);
            XY_CUDA(cudaMemcpyAsync(E.data(), pt->E_slot, SR * sizeof(double), cudaMemcpyDeviceToHost, pt->stream));
            XY_CUDA(cudaMemcpyAsync(M.data(), pt->M_slot, SR * 2 * sizeof(double), cudaMemcpyDeviceToHost, pt->stream));
            XY_CUDA(cudaMemcpyAsync(tos.data(), pt->temp_of_slot, SR * sizeof(int32_t), cudaMemcpyDeviceToHost, pt->stream));
            XY_CUDA(cudaStreamSynchronize(pt->stream));
            for (int s = 0; s < S; ++s)
                for (int r = 0; r < R; ++r) {
                    const size_t i = static_cast<size_t>(s) * R + r;
                    double *o = out_host + (static_cast<size_t>(s) * R + tos[i]) * 3;
                    o[0] = E[i]; o[1] = M[2 * i]; o[2] = M[2 * i + 1];
                }
        } catch (const std::bad_alloc &) {
            return fail(XY_ENOMEM, "host allocation failed");
        }
    }
    return XY_OK;
}

int xy_measure_fourier(xy_pt *pt, double *out_host) {
    if (!check_pt(pt)) return fail(XY_EINVAL, "bad handle");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    const xy_graph *g = pt->g;
    if (!g->coords) return fail(XY_ESTATE, "xy_graph_set_coords has not been called");
    const int S = g->S, R = pt->R;
    xy::FourierArgs a;
    a.theta = pt->theta; a.coords = g->coords; a.tab1 = g->tab1; a.tab2 = g->tab2;
    a.fk = pt->fk; a.ticket = pt->ticket; a.temp_of_slot = pt->temp_of_slot;
    a.G_slot = pt->G_slot; a.acc_k = pt->acc_k; a.N = g->N; a.R = R; a.s0 = 0;
    // two waves of 4 CTAs per SM over all samples and column blocks (measured on config 4: one wave 194 us, two 114 us,
    // three 127 us), at least 32 sites per warp, and at most 224 rows per warp: k_fourier2 flushes its fp32 partial sums
    // with same-address atomics after 256 rows, which a warp's range should never reach
    const int cb = pt->fast_G ? pt->col_blocks : 1;
    const int spw = pt->fast_G ? 32 / pt->fast_G : 1;
    const int warps_per_sample = std::max(1, std::min(ceil_div(g->N, 32), std::max(ceil_div(g->N, 224 * spw),
                                                                                   g->n_sm * 8 * xy::kWarps / (S * cb))));
    a.sites_per_warp = ceil_div(g->N, warps_per_sample);
    const dim3 grid(ceil_div(ceil_div(g->N, a.sites_per_warp), xy::kWarps), S, cb);
    // bulk-copy flavour (TMA fills the ring): needs 16-byte aligned rows -- G >= 2 and a 16-byte aligned theta
    const bool bulk = pt->fast_G >= 2 && (reinterpret_cast<uintptr_t>(pt->theta) & 15u) == 0;
#define XY_FOURIER2(GG)                                                                                     \
    case GG:                                                                                                \
        if (bulk) xy::k_fourier2<GG, (GG >= 2)><<<grid, xy::kBlock, xy::kFourierSmem, pt->stream>>>(a);     \
        else xy::k_fourier2<GG, false><<<grid, xy::kBlock, xy::kFourierSmem, pt->stream>>>(a);              \
        break;
    switch (pt->fast_G) {
        XY_FOURIER2(32) XY_FOURIER2(16) XY_FOURIER2(8) XY_FOURIER2(4) XY_FOURIER2(2) XY_FOURIER2(1)
        default: xy::k_fourier<<<grid, xy::kBlock, 0, pt->stream>>>(a); break;      // any R
    }
#undef XY_FOURIER2
    XY_CUDA(cudaGetLastError());
    pt->launches += 1;
    if (out_host) {
        const size_t SR = static_cast<size_t>(S) * R;
        try {
            std::vector<double> G(SR * 2);
            std::vector<int32_t> tos(SR);
            XY_CUDA(cudaMemcpyAsync(G.data(), pt->G_slot, SR * 2 * sizeof(double), cudaMemcpyDeviceToHost, pt->stream));
            XY_CUDA(cudaMemcpyAsync(tos.data(), pt->temp_of_slot, SR * sizeof(int32_t), cudaMemcpyDeviceToHost, pt->stream));
            XY_CUDA(cudaStreamSynchronize(pt->stream));
            for (int s = 0; s < S; ++s)
                for (int r = 0; r < R; ++r) {
                    const size_t i = static_cast<size_t>(s) * R + r;
                    double *o = out_host + (static_cast<size_t>(s) * R + tos[i]) * 2;
                    o[0] = G[2 * i]; o[1] = G[2 * i + 1];
                }
        } catch (const std::bad_alloc &) {
            return fail(XY_ENOMEM, "host allocation failed");
        }
    }
    return XY_OK;
}

int xy_read_fourier_accumulators(xy_pt *pt, double *acc_host) {
    if (!check_pt(pt) || !acc_host) return fail(XY_EINVAL, "bad handle or NULL buffer");
    DeviceGuard guard(pt->g->device);
    const size_t n = static_cast<size_t>(pt->g->S) * pt->R * 3;
    XY_CUDA(cudaMemcpyAsync(acc_host, pt->acc_k, n * sizeof(double), cudaMemcpyDeviceToHost, pt->stream));
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    return XY_OK;
}

int xy_set_schedule(xy_pt *pt, int samples_per_group) {
    if (!check_pt(pt) || samples_per_group < 0) return fail(XY_EINVAL, "bad handle or samples_per_group < 0");
    DeviceGuard guard(pt->g->device);
    pt->samples_per_group = samples_per_group;
    return XY_OK;
}

int xy_set_path(xy_pt *pt, int path) {
    if (!check_pt(pt) || path < 0 || path > 2) return fail(XY_EINVAL, "bad handle or path not in {0, 1, 2}");
    if (path == 2 && !cycle_eligible(pt, 1))
        return fail(XY_ESTATE, "the cluster path needs R = 2 * 2^k <= 64, fused measurement, samples whose rows fit the warps' "
                               "resident pools (shared memory), at most 12 colours and degrees <= 255");
    pt->path = path;
    return XY_OK;
}

int xy_get_path(xy_pt *pt, int or_per_sweep, int *path, int *cluster_size) {
    if (!check_pt(pt)) return fail(XY_EINVAL, "bad handle");
    const bool cyc = use_cycle_path(pt, or_per_sweep);
    if (path) *path = cyc ? 2 : 1;
    if (cluster_size) *cluster_size = cyc ? pt->cycle_C : 0;
    return XY_OK;
}

int xy_get_schedule(xy_pt *pt, int *samples_per_group, int64_t *group_bytes) {
    if (!check_pt(pt)) return fail(XY_EINVAL, "bad handle");
    const int group = auto_group(pt);
    if (samples_per_group) *samples_per_group = group;
    if (group_bytes)
        *group_bytes = static_cast<int64_t>(group) * (static_cast<int64_t>(pt->g->N) * pt->R * 4 + static_cast<int64_t>(pt->g->bytes_per_sample));
    return XY_OK;
}

int xy_set_tuning(xy_pt *pt, int balance, int pdl, int l2_persist, int fuse_measure, int cta_shape) {
    if (!check_pt(pt) || cta_shape < 0 || cta_shape > 2) return fail(XY_EINVAL, "bad handle or cta_shape not in {0, 1, 2}");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    pt->cta_shape = cta_shape;
    pt->balance = balance ? 1 : 0; pt->pdl = pdl ? 1 : 0; pt->l2_persist = l2_persist ? 1 : 0;
    pt->fuse_measure = fuse_measure ? 1 : 0;
    drop_graphs(pt);
    return XY_OK;
}

int xy_run(xy_pt *pt, int n_cycles, int sps, int orps, int me) {
    if (!check_pt(pt) || n_cycles < 0 || sps < 1 || orps < 0 || me < 0)
        return fail(XY_EINVAL, "need n_cycles >= 0, sweeps_per_swap >= 1, or_per_sweep >= 0, measure_every >= 0");
    DeviceGuard guard(pt->g->device);
    if (pt->order == 1 && orps != 1) return fail(XY_EINVAL, "the interleaved order needs or_per_sweep == 1");
    if (pt->path == 2 && !cycle_eligible(pt, orps))
        return fail(XY_ESTATE, "xy_set_path(2): the cluster path needs R = 2 * 2^k <= 64, or_per_sweep >= 1, fused measurement and samples that fit its resident pools");
    if (use_cycle_path(pt, orps)) {          // small samples: all cycles in one launch, one cluster per sample
        int rc = settle_upload(pt);
        if (rc == XY_OK) rc = launch_cycle(pt, n_cycles, sps, orps, me, true);
        if (rc != XY_OK) return rc;
        pt->sweep += static_cast<uint32_t>(n_cycles) * static_cast<uint32_t>(sps);
        pt->round += static_cast<uint32_t>(n_cycles);
        if (n_cycles > 0) pt->e_fresh = false;
        return XY_OK;
    }
    const int group = auto_group(pt);
    {
        const int rc = prepare_partitions(pt, group);
        if (rc != XY_OK) return rc;
    }
    if (pt->upload_armed && (n_cycles == 0 || group != pt->upload_group)) {
        const int rc = settle_upload(pt);
        if (rc != XY_OK) return rc;
    }
    for (int c = 0; c < n_cycles; ++c) {
        const int phase = me > 0 ? static_cast<int>(pt->sweep % static_cast<uint32_t>(me)) : 0;
        const bool await_upload = pt->upload_armed;      // first cycle after xy_set_theta_async: wait group by group
        pt->upload_armed = false;
        const CycleKey key{sps, orps, me, phase, group, await_upload ? 1 : 0};
        CycleGraph *cg = nullptr;
        const int rc = cached_graph(pt, key, [&] { return issue_cycle(pt, sps, orps, me, phase, group, await_upload); }, &cg);
        if (rc != XY_OK) return rc;
        XY_CUDA(cudaGraphLaunch(cg->exec, pt->stream));
        pt->launches += cg->launches;
        pt->sweep += static_cast<uint32_t>(sps);
        pt->round += 1;
        pt->e_fresh = false;  // labels moved; E per slot is still valid but keep the rule simple
    }
    return XY_OK;
}

int xy_run_sweeps(xy_pt *pt, int n_blocks, int sps, int orps) {
    if (!check_pt(pt) || n_blocks < 0 || sps < 1 || orps < 0)
        return fail(XY_EINVAL, "need n_blocks >= 0, sweeps_per_block >= 1, or_per_sweep >= 0");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    if (pt->order == 1 && orps != 1) return fail(XY_EINVAL, "the interleaved order needs or_per_sweep == 1");
    if (pt->path == 2 && !cycle_eligible(pt, orps))
        return fail(XY_ESTATE, "xy_set_path(2): the cluster path needs R = 2 * 2^k <= 64, or_per_sweep >= 1, fused measurement and samples that fit its resident pools");
    if (use_cycle_path(pt, orps)) {
        const int rc = launch_cycle(pt, n_blocks, sps, orps, 0, false);
        if (rc != XY_OK) return rc;
        pt->sweep += static_cast<uint32_t>(n_blocks) * static_cast<uint32_t>(sps);
        if (n_blocks > 0) pt->e_fresh = false;
        return XY_OK;
    }
    const int group = auto_group(pt);
    {
        const int rc = prepare_partitions(pt, group);
        if (rc != XY_OK) return rc;
    }
    for (int b = 0; b < n_blocks; ++b) {
        const CycleKey key{sps, orps, -1, 0, group, 0};
        CycleGraph *cg = nullptr;
        const int rc = cached_graph(pt, key, [&] { return issue_sweeps(pt, sps, orps, group); }, &cg);
        if (rc != XY_OK) return rc;
        XY_CUDA(cudaGraphLaunch(cg->exec, pt->stream));
        pt->launches += cg->launches;
        pt->sweep += static_cast<uint32_t>(sps);
        pt->e_fresh = false;
    }
    return XY_OK;
}

int xy_get_theta(xy_pt *pt, float *theta_host) {
    if (!check_pt(pt) || !theta_host) return fail(XY_EINVAL, "bad handle or NULL buffer");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    const size_t n = static_cast<size_t>(pt->g->S) * pt->g->N * pt->R;
    XY_CUDA(cudaMemcpyAsync(theta_host, pt->theta, n * sizeof(float), cudaMemcpyDeviceToHost, pt->stream));
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    return XY_OK;
}

int xy_set_theta(xy_pt *pt, const float *theta_host) {
    if (!check_pt(pt) || !theta_host) return fail(XY_EINVAL, "bad handle or NULL buffer");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    const size_t n = static_cast<size_t>(pt->g->S) * pt->g->N * pt->R;
    XY_CUDA(cudaMemcpyAsync(pt->theta, theta_host, n * sizeof(float), cudaMemcpyHostToDevice, pt->stream));
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    pt->e_fresh = false;
    return XY_OK;
}

int xy_set_theta_async(xy_pt *pt, const float *theta_host) {
    if (!check_pt(pt) || !theta_host) return fail(XY_EINVAL, "bad handle or NULL buffer");
    DeviceGuard guard(pt->g->device);
    const int S = pt->g->S, group = auto_group(pt);
    const size_t per_sample = static_cast<size_t>(pt->g->N) * pt->R;
    if (!pt->copy_stream) XY_CUDA(cudaStreamCreateWithFlags(&pt->copy_stream, cudaStreamNonBlocking));
    if (!pt->compute_done) XY_CUDA(cudaEventCreateWithFlags(&pt->compute_done, cudaEventDisableTiming));
    const size_t n_groups = static_cast<size_t>((S + group - 1) / group);
    if (pt->upload_group != group || pt->upload_ev.size() != n_groups) {
        XY_CUDA(cudaStreamSynchronize(pt->stream));      // graphs that wait on the old events must have finished
        drop_graphs(pt);
        for (cudaEvent_t ev : pt->upload_ev) cudaEventDestroy(ev);
        pt->upload_ev.clear();
        for (size_t k = 0; k < n_groups; ++k) {
            cudaEvent_t ev = nullptr;
            XY_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
            pt->upload_ev.push_back(ev);
        }
        pt->upload_group = group;
    }
    // the uploads overwrite theta: they start after everything already enqueued on the compute stream
    XY_CUDA(cudaEventRecord(pt->compute_done, pt->stream));
    XY_CUDA(cudaStreamWaitEvent(pt->copy_stream, pt->compute_done, 0));
    for (int s0 = 0; s0 < S; s0 += group) {
        const int s1 = std::min(S, s0 + group);
        XY_CUDA(cudaMemcpyAsync(pt->theta + s0 * per_sample, theta_host + s0 * per_sample, (s1 - s0) * per_sample * sizeof(float),
                                cudaMemcpyHostToDevice, pt->copy_stream));
        XY_CUDA(cudaEventRecord(pt->upload_ev[s0 / group], pt->copy_stream));
    }
    pt->upload_armed = true;
    pt->e_fresh = false;
    return XY_OK;
}

int xy_get_labels(xy_pt *pt, int32_t *temp_of_slot_host) {
    if (!check_pt(pt) || !temp_of_slot_host) return fail(XY_EINVAL, "bad handle or NULL buffer");
    DeviceGuard guard(pt->g->device);
    const size_t SR = static_cast<size_t>(pt->g->S) * pt->R;
    XY_CUDA(cudaMemcpyAsync(temp_of_slot_host, pt->temp_of_slot, SR * sizeof(int32_t), cudaMemcpyDeviceToHost, pt->stream));
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    return XY_OK;
}

int xy_set_labels(xy_pt *pt, const int32_t *temp_of_slot_host) {
    if (!check_pt(pt) || !temp_of_slot_host) return fail(XY_EINVAL, "bad handle or NULL buffer");
    DeviceGuard guard(pt->g->device);
    const int S = pt->g->S, R = pt->R;
    try {
        std::vector<uint8_t> seen(R);
        for (int s = 0; s < S; ++s) {
            std::fill(seen.begin(), seen.end(), 0);
            for (int r = 0; r < R; ++r) {
                const int t = temp_of_slot_host[static_cast<size_t>(s) * R + r];
                if (t < 0 || t >= R || seen[t]) return fail(XY_EINVAL, "labels are not a permutation of 0..R-1");
                seen[t] = 1;
            }
        }
    } catch (const std::bad_alloc &) {
        return fail(XY_ENOMEM, "host allocation failed");
    }
    const size_t SR = static_cast<size_t>(S) * R;
    XY_CUDA(cudaMemcpyAsync(pt->temp_of_slot, temp_of_slot_host, SR * sizeof(int32_t), cudaMemcpyHostToDevice, pt->stream));
    xy::k_refresh_slot_params<<<ceil_div(SR, 128), 128, 0, pt->stream>>>(pt->temp_of_slot, pt->slot_of_temp, pt->beta_f, pt->w_f,
                                                                        pt->beta_slot, pt->w_slot, S, R);
    XY_CUDA(cudaGetLastError());
    pt->launches += 1;
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    return XY_OK;
}

int xy_get_energy(xy_pt *pt, double *E_slot_host) {
    if (!check_pt(pt) || !E_slot_host) return fail(XY_EINVAL, "bad handle or NULL buffer");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    if (!pt->e_fresh) {
        const int rc = launch_measure(pt, 0, pt->g->S, false);
        if (rc != XY_OK) return rc;
        pt->e_fresh = true;
    }
    const size_t SR = static_cast<size_t>(pt->g->S) * pt->R;
    XY_CUDA(cudaMemcpyAsync(E_slot_host, pt->E_slot, SR * sizeof(double), cudaMemcpyDeviceToHost, pt->stream));
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    return XY_OK;
}

int xy_read_accumulators(xy_pt *pt, double *acc_host) {
    if (!check_pt(pt) || !acc_host) return fail(XY_EINVAL, "bad handle or NULL buffer");
    DeviceGuard guard(pt->g->device);
    const size_t n = static_cast<size_t>(pt->g->S) * pt->R * XY_NACC;
    XY_CUDA(cudaMemcpyAsync(acc_host, pt->acc, n * sizeof(double), cudaMemcpyDeviceToHost, pt->stream));
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    return XY_OK;
}

int xy_reset_accumulators(xy_pt *pt) {
    if (!check_pt(pt)) return fail(XY_EINVAL, "bad handle");
    DeviceGuard guard(pt->g->device);
    const size_t n = static_cast<size_t>(pt->g->S) * pt->R * XY_NACC;
    XY_CUDA(cudaMemsetAsync(pt->acc, 0, n * sizeof(double), pt->stream));
    XY_CUDA(cudaMemsetAsync(pt->acc_k, 0, static_cast<size_t>(pt->g->S) * pt->R * 3 * sizeof(double), pt->stream));
    return XY_OK;
}

int xy_get_counters(xy_pt *pt, uint32_t *sweep, uint32_t *round, int64_t *att, int64_t *acc) {
    if (!check_pt(pt)) return fail(XY_EINVAL, "bad handle");
    DeviceGuard guard(pt->g->device);
    uint32_t c[2];
    const size_t SR = static_cast<size_t>(pt->g->S) * pt->R;
    XY_CUDA(cudaMemcpyAsync(c, pt->counters, sizeof(c), cudaMemcpyDeviceToHost, pt->stream));
    if (att) XY_CUDA(cudaMemcpyAsync(att, pt->attempts, SR * sizeof(int64_t), cudaMemcpyDeviceToHost, pt->stream));
    if (acc) XY_CUDA(cudaMemcpyAsync(acc, pt->accepts, SR * sizeof(int64_t), cudaMemcpyDeviceToHost, pt->stream));
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    if (c[0] != pt->sweep || c[1] != pt->round) return fail(XY_ESTATE, "device counters diverged from the host mirror");
    if (sweep) *sweep = c[0];
    if (round) *round = c[1];
    return XY_OK;
}

int xy_set_counters(xy_pt *pt, uint32_t sweep, uint32_t round) {
    if (!check_pt(pt)) return fail(XY_EINVAL, "bad handle");
    DeviceGuard guard(pt->g->device);
    const uint32_t c[2] = {sweep, round};
    XY_CUDA(cudaMemcpyAsync(pt->counters, c, sizeof(c), cudaMemcpyHostToDevice, pt->stream));
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    pt->sweep = sweep; pt->round = round;
    return XY_OK;
}

int xy_theta_device(xy_pt *pt, float **theta_dev) {
    if (!check_pt(pt) || !theta_dev) return fail(XY_EINVAL, "bad handle or NULL out");
    DeviceGuard guard(pt->g->device);
    *theta_dev = pt->theta;
    return XY_OK;
}

int xy_launch_count(xy_pt *pt, int64_t *n) {
    if (!check_pt(pt) || !n) return fail(XY_EINVAL, "bad handle or NULL out");
    DeviceGuard guard(pt->g->device);
    *n = pt->launches;
    return XY_OK;
}

int xy_l2_bandwidth(size_t bytes, int mode, int repeats, void *stream, double *gbs_out) {
    if (!gbs_out || bytes < (1u << 20) || bytes > (size_t(1) << 32) || mode < 0 || mode > 1 || repeats < 1)
        return fail(XY_EINVAL, "need 1 MiB <= bytes <= 4 GiB, mode in {0, 1}, repeats >= 1, non-NULL output");
    int dev = 0, n_sm = 0;
    XY_CUDA(cudaGetDevice(&dev));
    XY_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    size_t n_rows = 1;                                      // 256-byte rows: the largest power of two that fits
    while (n_rows * 2 * 256 <= bytes) n_rows *= 2;
    const int grid = n_sm * 4, threads = 512, passes = 16;
    const size_t n_vec = bytes / 16 / grid;                  // uint4 per CTA slice (stream mode)
    const size_t moved = mode == 0 ? n_vec * 16 * grid * passes : n_rows * 256 * passes;
    const int rows_per_warp = static_cast<int>((n_rows * passes / (static_cast<size_t>(grid) * (threads / 32)) + 7) / 8 * 8);
    unsigned char *buf = nullptr;
    unsigned *sink = nullptr;
    int rc;
    if ((rc = dev_alloc(&buf, bytes)) != XY_OK) return rc;
    if ((rc = dev_alloc(&sink, 1)) != XY_OK) { cudaFree(buf); return rc; }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaMemsetAsync(buf, 0, bytes, st);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    double best = 0.0;
    for (int r = 0; r < repeats + 2 && e == cudaSuccess; ++r) {       // two untimed launches warm L2 and the clocks
        e = cudaEventRecord(e0, st);
        if (e != cudaSuccess) break;
        if (mode == 0) xy::k_l2_stream<<<grid, threads, 0, st>>>(reinterpret_cast<const uint4 *>(buf), n_vec, passes, sink);
        else xy::k_l2_gather<<<grid, threads, 0, st>>>(reinterpret_cast<const uint2 *>(buf), static_cast<uint32_t>(n_rows), rows_per_warp, sink);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventRecord(e1, st);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        const double bytes_done = mode == 0 ? static_cast<double>(moved)
                                            : static_cast<double>(rows_per_warp) * grid * (threads / 32) * 256.0;
        if (e == cudaSuccess && r >= 2 && ms > 0.f) best = std::max(best, bytes_done / (ms * 1e-3) * 1e-9);
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf); cudaFree(sink);
    if (e != cudaSuccess) return fail(XY_ECUDA, std::string("xy_l2_bandwidth: ") + cudaGetErrorString(e));
    *gbs_out = best;
    return XY_OK;
}

int xy_synchronize(xy_pt *pt) {
    if (!check_pt(pt)) return fail(XY_EINVAL, "bad handle");
    DeviceGuard guard(pt->g->device);
    { const int rc_up = settle_upload(pt); if (rc_up != XY_OK) return rc_up; }
    XY_CUDA(cudaStreamSynchronize(pt->stream));
    return XY_OK;
}

}  // extern "C"
