// levy_graph.cpp -- host-side Levy-graph builder + smallest-last colouring (see include/xy_levy.h).
//
// Seeded input generator for both the CUDA path and the oracle-driven tests.  Fast data structures
// (CDF table + binary search, open-addressing edge set, ordered-set smallest-last queue); the
// definition-level restatement it is checked against lives in the oracle directory and shares no code
// with this file.  PAPER.md:31, :96-103 (Eq. 6), :452-456 (App. B.a), :490 (colour-sorted storage).
#include "xy_levy.h"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <set>
#include <string>
#include <thread>
#include <utility>
#include <vector>

namespace {

thread_local std::string g_err;

int fail(int code, const std::string &msg) {
    g_err = msg;
    return code;
}

// Philox4x32-10, written from the published round function (Salmon et al., SC'11).
inline void philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                   uint32_t out[4]) {
    for (int r = 0; r < 10; ++r) {
        const uint64_t a = 0xD2511F53ull * c0, b = 0xCD9E8D57ull * c2;
        const uint32_t n0 = static_cast<uint32_t>(b >> 32) ^ c1 ^ k0;
        const uint32_t n2 = static_cast<uint32_t>(a >> 32) ^ c3 ^ k1;
        c1 = static_cast<uint32_t>(b);
        c3 = static_cast<uint32_t>(a);
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// open-addressing set of undirected bonds keyed by (min<<32 | max)
class BondSet {
public:
    explicit BondSet(size_t n_expected) {
        size_t cap = 16;
        while (cap < 2 * n_expected + 8) cap <<= 1;
        slots_.assign(cap, kEmpty);
        mask_ = cap - 1;
    }
    bool insert(uint32_t a, uint32_t b) {  // false if already present
        const uint64_t key = (static_cast<uint64_t>(std::min(a, b)) << 32) | std::max(a, b);
        size_t h = static_cast<size_t>((key * 0x9E3779B97F4A7C15ull) >> 20) & mask_;
        while (slots_[h] != kEmpty) {
            if (slots_[h] == key) return false;
            h = (h + 1) & mask_;
        }
        slots_[h] = key;
        return true;
    }
private:
    static constexpr uint64_t kEmpty = ~0ull;
    std::vector<uint64_t> slots_;
    size_t mask_ = 0;
};

void csr_from_bonds(int N, const std::vector<std::pair<int32_t, int32_t>> &bonds,
                    std::vector<int32_t> &row_ptr, std::vector<int32_t> &col_idx) {
    row_ptr.assign(static_cast<size_t>(N) + 1, 0);
    for (const auto &e : bonds) { row_ptr[e.first + 1]++; row_ptr[e.second + 1]++; }
    for (int i = 0; i < N; ++i) row_ptr[i + 1] += row_ptr[i];
    col_idx.resize(static_cast<size_t>(row_ptr[N]));
    std::vector<int32_t> fill(row_ptr.begin(), row_ptr.end() - 1);
    for (const auto &e : bonds) {
        col_idx[fill[e.first]++] = e.second;
        col_idx[fill[e.second]++] = e.first;
    }
    for (int i = 0; i < N; ++i) std::sort(col_idx.begin() + row_ptr[i], col_idx.begin() + row_ptr[i + 1]);
}

// smallest-last ordering with exact (degree, id) tie-breaking, then greedy colouring
int colour_sl(int N, const int32_t *row_ptr, const int32_t *col_idx, int32_t *colour) {
    std::vector<int32_t> deg(N), order(N);
    std::vector<uint8_t> removed(N, 0);
    std::set<std::pair<int32_t, int32_t>> queue;
    for (int v = 0; v < N; ++v) {
        deg[v] = row_ptr[v + 1] - row_ptr[v];
        queue.emplace_hint(queue.end(), deg[v], v);
    }
    // emplace_hint with end() is only a hint; the set orders by (deg, id) regardless
    for (int step = N - 1; step >= 0; --step) {
        const auto it = queue.begin();
        const int v = it->second;
        queue.erase(it);
        order[step] = v;
        removed[v] = 1;
        for (int e = row_ptr[v]; e < row_ptr[v + 1]; ++e) {
            const int u = col_idx[e];
            if (removed[u]) continue;
            queue.erase({deg[u], u});
            --deg[u];
            queue.emplace(deg[u], u);
        }
    }
    std::fill(colour, colour + N, -1);
    int Q = 0;
    std::vector<int32_t> mark;  // mark[c] == v  <=> colour c is used by a neighbour of v
    for (int step = 0; step < N; ++step) {
        const int v = order[step];
        for (int e = row_ptr[v]; e < row_ptr[v + 1]; ++e) {
            const int c = colour[col_idx[e]];
            if (c >= 0) {
                if (static_cast<size_t>(c) >= mark.size()) mark.resize(c + 1, -1);
                mark[c] = v;
            }
        }
        int c = 0;
        while (static_cast<size_t>(c) < mark.size() && mark[c] == v) ++c;
        colour[v] = c;
        Q = std::max(Q, c + 1);
    }
    return Q;
}

// Shrink (ideally: empty) the LAST colour class of a proper colouring with Q colours.  Smallest-last leaves ~1.4 % of
// the sites in a fifth class at z = 6: a fifth sequential phase per sweep for almost no work (PAPER.md:456 Q, :494
// time ~ Q/2).  The Levy graphs of the configs with rho >= 3 contain a few 5-cliques, so the fifth colour cannot go
// away there -- but it is needed by a handful of sites, not by thousands.
// Tabu / min-conflicts search: the sites of the last class (colour T = Q-1) take the least conflicting of the other
// colours; then, while monochromatic bonds remain, a conflicting site (picked by the Philox stream of domain 5) moves
// to its least conflicting colour < T that is not tabu (aspiration: a conflict-free colour is always allowed) and may
// not move back for a few steps.  After max_moves such moves, at a moment when the search is near the fewest bad bonds
// it has seen, the escape opens: a conflicting site without a conflict-free colour returns to colour T if none of its
// neighbours holds it (late in the search such neighbours are pushed back below T first).  When no bad bond is left, sites of colour T that have a free colour leave it
// again.  Returns T if the last class is empty (the graph is T-coloured), else Q with a proper Q-colouring whose last
// class is small; if that is not smaller than the input's, or bad bonds remain after 4 max_moves moves, colour[] is
// left untouched.  Deterministic in (graph, seed, sample).
int colour_reduce_once(int N, const int32_t *row_ptr, const int32_t *col_idx, int32_t *colour, int Q, uint64_t seed,
                       uint32_t sample, int64_t max_moves) {
    if (Q < 3) return Q;
    const int T = Q - 1;
    std::vector<int32_t> col(colour, colour + N);
    std::vector<int32_t> cnt(static_cast<size_t>(N) * Q, 0);      // cnt[v*Q + c] = neighbours of v with colour c
    auto at = [&](int v, int c) -> int32_t & { return cnt[static_cast<size_t>(v) * Q + c]; };
    auto bump = [&](int v, int c, int d) {
        for (int e = row_ptr[v]; e < row_ptr[v + 1]; ++e) at(col_idx[e], c) += d;
    };
    int64_t last_class = 0;
    for (int v = 0; v < N; ++v) {
        if (col[v] < T) bump(v, col[v], +1);
        else ++last_class;
    }
    for (int v = 0; v < N; ++v) {
        if (col[v] < T) continue;
        int best = 0;
        for (int c = 1; c < T; ++c)
            if (at(v, c) < at(v, best)) best = c;
        col[v] = best;
        bump(v, best, +1);
    }
    std::vector<int32_t> conf, where(N, -1);                       // the conflicting sites, and their position in conf
    auto refresh = [&](int v) {
        const bool bad = at(v, col[v]) > 0;
        if (bad && where[v] < 0) { where[v] = static_cast<int32_t>(conf.size()); conf.push_back(v); }
        else if (!bad && where[v] >= 0) {
            const int32_t last = conf.back();
            conf[where[v]] = last; where[last] = where[v];
            conf.pop_back(); where[v] = -1;
        }
    };
    auto move = [&](int v, int c) {
        bump(v, col[v], -1);
        col[v] = c;
        bump(v, c, +1);
        refresh(v);
        for (int e = row_ptr[v]; e < row_ptr[v + 1]; ++e) refresh(col_idx[e]);
    };
    for (int v = 0; v < N; ++v) refresh(v);
    std::vector<int64_t> tabu(static_cast<size_t>(N) * T, -1);     // move (v -> c) forbidden while it <= tabu
    const uint32_t k0 = static_cast<uint32_t>(seed), k1 = static_cast<uint32_t>(seed >> 32);
    size_t fewest = conf.size();                                   // fewest conflicting sites seen so far
    bool escape = false;
    for (int64_t it = 0; !conf.empty(); ++it) {
        if (it >= 4 * max_moves) return Q;
        fewest = std::min(fewest, conf.size());
        // the escape opens after max_moves moves, at a moment when the search is (again) near its best state
        if (!escape && (it >= 2 * max_moves || (it >= max_moves && conf.size() <= fewest + fewest / 8 + 1))) escape = true;
        uint32_t x[4];
        philox(static_cast<uint32_t>(it), static_cast<uint32_t>(static_cast<uint64_t>(it) >> 32), sample, 5u, k0, k1, x);
        const int v = conf[(static_cast<uint64_t>(x[0]) * conf.size()) >> 32];
        const int old = col[v];
        int best = -1, n_best = 0;
        for (int c = 0; c < T; ++c) {
            if (c == old) continue;
            const int32_t k = at(v, c);
            if (tabu[static_cast<size_t>(v) * T + c] >= it && k > 0) continue;
            if (best < 0 || k < at(v, best)) { best = c; n_best = 1; }
            else if (k == at(v, best) && ((x[1] >> (n_best++ & 15)) & 1u)) best = c;
        }
        if (escape && (best < 0 || at(v, best) > 0) && (at(v, T) == 0 || it >= 3 * max_moves)) {
            // no conflict-free colour: v takes the last colour; late in the search, neighbours that hold it are pushed
            // back to their least conflicting colour below T first (they may become conflicting sites themselves)
            for (int e = row_ptr[v]; e < row_ptr[v + 1] && at(v, T) > 0; ++e) {
                const int u = col_idx[e];
                if (col[u] != T) continue;
                int bu = 0;
                for (int c = 1; c < T; ++c)
                    if (at(u, c) < at(u, bu)) bu = c;
                move(u, bu);
            }
            move(v, T);
            continue;
        }
        if (best < 0) continue;                                    // every other colour is tabu: draw again
        tabu[static_cast<size_t>(v) * T + old] = it + 8 + (x[2] & 7u);
        move(v, best);
    }
    int64_t left = 0;
    for (int v = 0; v < N; ++v) {
        if (col[v] < T) continue;
        int c = 0;
        while (c < T && at(v, c) > 0) ++c;
        if (c < T) move(v, c);
        else ++left;
    }
    if (left >= last_class) return Q;                              // no gain: keep the input
    std::copy(col.begin(), col.end(), colour);
    return left == 0 ? T : Q;
}

// colour_reduce_once until the number of colours reaches target_q or the last class stops shrinking (at most 8 rounds;
// round r uses the Philox stream of sample + r * 2^16 so that a repeated search does not retrace the previous one)
int colour_reduce(int N, const int32_t *row_ptr, const int32_t *col_idx, int32_t *colour, int Q, int target_q, uint64_t seed,
                  uint32_t sample, int64_t max_moves) {
    auto last_size = [&](int q) {
        int64_t n = 0;
        for (int v = 0; v < N; ++v) n += colour[v] == q - 1;
        return n;
    };
    int64_t size = last_size(Q);
    for (uint32_t round = 0; round < 8 && Q > target_q; ++round) {
        const int q2 = colour_reduce_once(N, row_ptr, col_idx, colour, Q, seed, sample + (round << 16), max_moves);
        const int64_t size2 = last_size(q2);
        if (q2 == Q && size2 >= size) break;
        Q = q2;
        size = size2;
    }
    return Q;
}

void renumber(int N, const int32_t *row_ptr, const int32_t *col_idx, const int32_t *colour,
              int32_t *new_to_old, int32_t *row_ptr_new, int32_t *col_idx_new, int32_t *colour_new) {
    std::vector<int32_t> n2o(N), o2n(N);
    for (int v = 0; v < N; ++v) n2o[v] = v;
    std::stable_sort(n2o.begin(), n2o.end(), [&](int a, int b) { return colour[a] < colour[b]; });
    for (int a = 0; a < N; ++a) o2n[n2o[a]] = a;
    row_ptr_new[0] = 0;
    for (int a = 0; a < N; ++a) {
        const int v = n2o[a];
        const int n = row_ptr[v + 1] - row_ptr[v];
        int32_t *row = col_idx_new + row_ptr_new[a];
        for (int q = 0; q < n; ++q) row[q] = o2n[col_idx[row_ptr[v] + q]];
        std::sort(row, row + n);
        row_ptr_new[a + 1] = row_ptr_new[a] + n;
        colour_new[a] = colour[v];
    }
    if (new_to_old) std::copy(n2o.begin(), n2o.end(), new_to_old);
}

struct Cdf {
    std::vector<double> run;  // run[d] = sum_{d'=1..d} w_d', run[0] = 0
    double total = 0.0;
    bool fbc = false;         // free boundaries: displacements (dx, dy) in [-(L-1), L-1]^2, plain Euclidean distance
};

// free boundary conditions (r up to L sqrt 2): run[] over the (2L-1)^2 displacement vectors in index
// order d = (dy + L-1)(2L-1) + (dx + L-1) + 1, the null vector has weight 0 (DESIGN R21)
Cdf make_cdf_fbc(int L, double rho) {
    const int W = 2 * L - 1;
    Cdf c;
    c.fbc = true;
    c.run.assign(static_cast<size_t>(W) * W + 1, 0.0);
    double s = 0.0;
    for (int d = 0; d < W * W; ++d) {
        const int dx = d % W - (L - 1), dy = d / W - (L - 1);
        if (dx != 0 || dy != 0) s += std::pow(static_cast<double>(dx * dx + dy * dy), -0.5 * rho);
        c.run[static_cast<size_t>(d) + 1] = s;
    }
    c.total = s;
    return c;
}

Cdf make_cdf(int L, double rho) {
    const int N = L * L;
    Cdf c;
    c.run.assign(static_cast<size_t>(N), 0.0);
    double s = 0.0;
    for (int d = 1; d < N; ++d) {
        const int dx = d % L, dy = d / L;
        const int mx = std::min(dx, L - dx), my = std::min(dy, L - dy);
        s += std::pow(static_cast<double>(mx * mx + my * my), -0.5 * rho);
        c.run[d] = s;
    }
    c.total = s;
    return c;
}

int build_one(int L, int z, uint64_t seed, uint32_t sample, const Cdf &cdf, int reduce_moves_per_site, int32_t *row_ptr,
              int32_t *col_idx, int32_t *colour, int32_t *new_to_old, int32_t *n_colours,
              int64_t *n_draws, std::string &err) {
    const int N = L * L;
    const int64_t n_bonds = static_cast<int64_t>(N) * z / 2;
    const int64_t max_draws = 64 * n_bonds + (1ll << 22);
    std::vector<std::pair<int32_t, int32_t>> bonds;
    bonds.reserve(static_cast<size_t>(n_bonds));
    BondSet present(static_cast<size_t>(n_bonds));
    const uint32_t k0 = static_cast<uint32_t>(seed), k1 = static_cast<uint32_t>(seed >> 32);
    int64_t k = 0;
    while (static_cast<int64_t>(bonds.size()) < n_bonds) {
        if (k >= max_draws) { err = "draw limit reached (rho too large for this z?)"; return XY_LEVY_EDRAWS; }
        uint32_t x[4];
        philox(static_cast<uint32_t>(k), static_cast<uint32_t>(static_cast<uint64_t>(k) >> 32), sample, 3u, k0, k1, x);
        ++k;
        const int i = static_cast<int>((static_cast<uint64_t>(x[0]) * static_cast<uint64_t>(N)) >> 32);
        const uint64_t m53 = (static_cast<uint64_t>(x[1]) << 21) | (static_cast<uint64_t>(x[2]) >> 11);
        const double target = ((static_cast<double>(m53) + 0.5) * 1.1102230246251565e-16) * cdf.total;
        const int xi = i % L, yi = i / L;
        int j;
        if (cdf.fbc) {
            // first d in [1, W^2] with run[d] > target; displacement index d - 1; a partner outside the lattice
            // discards the whole draw (pairs are drawn with P ~ r^-rho among the pairs that exist)
            const int W = 2 * L - 1;
            int d = static_cast<int>(std::upper_bound(cdf.run.begin() + 1, cdf.run.end(), target) - cdf.run.begin());
            if (d > W * W) d = W * W;
            const int xj = xi + (d - 1) % W - (L - 1), yj = yi + (d - 1) / W - (L - 1);
            if (xj < 0 || xj >= L || yj < 0 || yj >= L || (xj == xi && yj == yi)) continue;
            j = yj * L + xj;
        } else {
            // first d in [1, N-1] with run[d] > target
            int d = static_cast<int>(std::upper_bound(cdf.run.begin() + 1, cdf.run.end(), target) - cdf.run.begin());
            if (d > N - 1) d = N - 1;
            j = ((yi + d / L) % L) * L + (xi + d % L) % L;
        }
        if (!present.insert(static_cast<uint32_t>(i), static_cast<uint32_t>(j))) continue;
        bonds.emplace_back(i, j);
    }
    std::vector<int32_t> rp, ci, col(N);
    csr_from_bonds(N, bonds, rp, ci);
    int Q = colour_sl(N, rp.data(), ci.data(), col.data());
    // optional: fewer colours / a smaller last class by local search (colour_reduce_once), down to 3 colours at most
    if (reduce_moves_per_site > 0) Q = colour_reduce(N, rp.data(), ci.data(), col.data(), Q, 3, seed, sample,
                                                     static_cast<int64_t>(reduce_moves_per_site) * N);
    renumber(N, rp.data(), ci.data(), col.data(), new_to_old, row_ptr, col_idx, colour);
    if (n_colours) *n_colours = Q;
    if (n_draws) *n_draws = k;
    return XY_LEVY_OK;
}

bool csr_ok(int N, const int32_t *row_ptr, const int32_t *col_idx) {
    if (N < 0 || !row_ptr || row_ptr[0] != 0) return false;
    for (int i = 0; i < N; ++i) if (row_ptr[i + 1] < row_ptr[i]) return false;
    if (row_ptr[N] > 0 && !col_idx) return false;
    for (int e = 0; e < row_ptr[N]; ++e) if (col_idx[e] < 0 || col_idx[e] >= N) return false;
    return true;
}

}  // namespace

extern "C" {

const char *xy_levy_last_error(void) { return g_err.c_str(); }

static int levy_build_impl(bool fbc, int reduce_moves_per_site, int L, double rho, int z, uint64_t seed, uint32_t sample_base,
                           int S, int n_threads, int32_t *row_ptr, int32_t *col_idx, int32_t *colour, int32_t *new_to_old,
                           int32_t *n_colours, int64_t *n_draws) {
    try {
        if (L < 2 || L > 16384 || z < 1 || S < 0 || !(rho >= 0.0) || !std::isfinite(rho))
            return fail(XY_LEVY_EINVAL, "need 2 <= L <= 16384, z >= 1, S >= 0, finite rho >= 0");
        const int64_t N = static_cast<int64_t>(L) * L;
        if ((N * z) % 2 != 0) return fail(XY_LEVY_EINVAL, "N*z must be even");
        if (N * z / 2 > N * (N - 1) / 2) return fail(XY_LEVY_EINVAL, "more bonds than pairs");
        if (N * z > 0x7fffffffll) return fail(XY_LEVY_EINVAL, "nnz exceeds int32");
        if (S > 0 && (!row_ptr || !col_idx || !colour)) return fail(XY_LEVY_EINVAL, "null output array");
        if (fbc && L > 2048) return fail(XY_LEVY_EINVAL, "free boundaries: L <= 2048");
        const Cdf cdf = fbc ? make_cdf_fbc(L, rho) : make_cdf(L, rho);
        if (!(cdf.total > 0.0) || !std::isfinite(cdf.total)) return fail(XY_LEVY_EINVAL, "degenerate weights");
        int nt = n_threads > 0 ? n_threads : static_cast<int>(std::thread::hardware_concurrency());
        nt = std::max(1, std::min(nt, S));
        std::atomic<int> next{0};
        std::atomic<int> status{XY_LEVY_OK};
        std::vector<std::string> errs(nt);
        auto work = [&](int tid) {
            try {
                for (int s = next.fetch_add(1); s < S; s = next.fetch_add(1)) {
                    const int rc = build_one(L, z, seed, sample_base + static_cast<uint32_t>(s), cdf, reduce_moves_per_site,
                                             row_ptr + static_cast<size_t>(s) * (N + 1),
                                             col_idx + static_cast<size_t>(s) * N * z,
                                             colour + static_cast<size_t>(s) * N,
                                             new_to_old ? new_to_old + static_cast<size_t>(s) * N : nullptr,
                                             n_colours ? n_colours + s : nullptr, n_draws ? n_draws + s : nullptr,
                                             errs[tid]);
                    if (rc != XY_LEVY_OK) { status.store(rc); return; }
                }
            } catch (const std::bad_alloc &) {
                errs[tid] = "out of memory";
                status.store(XY_LEVY_ENOMEM);
            }
        };
        std::vector<std::thread> pool;
        for (int t = 1; t < nt; ++t) pool.emplace_back(work, t);
        work(0);
        for (auto &t : pool) t.join();
        if (status.load() != XY_LEVY_OK) {
            std::string msg;
            for (const auto &e : errs) if (!e.empty()) msg = e;
            return fail(status.load(), msg);
        }
        return XY_LEVY_OK;
    } catch (const std::bad_alloc &) {
        return fail(XY_LEVY_ENOMEM, "out of memory");
    } catch (...) {
        return fail(XY_LEVY_EINVAL, "unexpected exception");
    }
}

int xy_levy_build(int L, double rho, int z, uint64_t seed, uint32_t sample_base, int S, int n_threads,
                  int32_t *row_ptr, int32_t *col_idx, int32_t *colour, int32_t *new_to_old,
                  int32_t *n_colours, int64_t *n_draws) {
    return levy_build_impl(false, 0, L, rho, z, seed, sample_base, S, n_threads, row_ptr, col_idx, colour, new_to_old,
                           n_colours, n_draws);
}

int xy_levy_build_fbc(int L, double rho, int z, uint64_t seed, uint32_t sample_base, int S, int n_threads,
                      int32_t *row_ptr, int32_t *col_idx, int32_t *colour, int32_t *new_to_old,
                      int32_t *n_colours, int64_t *n_draws) {
    return levy_build_impl(true, 0, L, rho, z, seed, sample_base, S, n_threads, row_ptr, col_idx, colour, new_to_old,
                           n_colours, n_draws);
}

int xy_levy_build_opt(int free_boundaries, int reduce_moves_per_site, int L, double rho, int z, uint64_t seed,
                      uint32_t sample_base, int S, int n_threads, int32_t *row_ptr, int32_t *col_idx, int32_t *colour,
                      int32_t *new_to_old, int32_t *n_colours, int64_t *n_draws) {
    if (reduce_moves_per_site < 0) return fail(XY_LEVY_EINVAL, "reduce_moves_per_site < 0");
    return levy_build_impl(free_boundaries != 0, reduce_moves_per_site, L, rho, z, seed, sample_base, S, n_threads, row_ptr,
                           col_idx, colour, new_to_old, n_colours, n_draws);
}

int xy_colour_smallest_last(int N, const int32_t *row_ptr, const int32_t *col_idx, int32_t *colour) {
    try {
        if (!csr_ok(N, row_ptr, col_idx) || (N > 0 && !colour)) return fail(XY_LEVY_EINVAL, "malformed CSR");
        return colour_sl(N, row_ptr, col_idx, colour);
    } catch (const std::bad_alloc &) {
        return fail(XY_LEVY_ENOMEM, "out of memory");
    }
}

int xy_colour_reduce(int N, const int32_t *row_ptr, const int32_t *col_idx, int32_t *colour, int target_q, uint64_t seed,
                     uint32_t sample, int64_t max_moves) {
    try {
        if (!csr_ok(N, row_ptr, col_idx) || (N > 0 && !colour) || target_q < 2 || max_moves < 0)
            return fail(XY_LEVY_EINVAL, "malformed CSR, null colour array, target_q < 2 or max_moves < 0");
        int Q = 0;
        for (int v = 0; v < N; ++v) {
            if (colour[v] < 0) return fail(XY_LEVY_EINVAL, "negative colour");
            Q = std::max(Q, colour[v] + 1);
        }
        for (int v = 0; v < N; ++v)
            for (int e = row_ptr[v]; e < row_ptr[v + 1]; ++e)
                if (colour[col_idx[e]] == colour[v]) return fail(XY_LEVY_EINVAL, "the input colouring is not proper");
        return colour_reduce(N, row_ptr, col_idx, colour, Q, target_q, seed, sample, max_moves);
    } catch (const std::bad_alloc &) {
        return fail(XY_LEVY_ENOMEM, "out of memory");
    }
}

int xy_renumber_colour_major(int N, const int32_t *row_ptr, const int32_t *col_idx, const int32_t *colour,
                             int32_t *new_to_old, int32_t *row_ptr_new, int32_t *col_idx_new,
                             int32_t *colour_new) {
    try {
        if (!csr_ok(N, row_ptr, col_idx) || (N > 0 && (!colour || !row_ptr_new || !colour_new)))
            return fail(XY_LEVY_EINVAL, "malformed CSR or null output");
        renumber(N, row_ptr, col_idx, colour, new_to_old, row_ptr_new, col_idx_new, colour_new);
        return XY_LEVY_OK;
    } catch (const std::bad_alloc &) {
        return fail(XY_LEVY_ENOMEM, "out of memory");
    }
}

}  // extern "C"
