/*
 * xy_oracle.c -- CPU ORACLE (test infrastructure, NOT the product; see xy_oracle.h).
 *
 * A plain, slow, single-threaded restatement of what the hot path of arXiv 1211.3991
 * computes: graph-coloured Metropolis + over-relaxation sweeps of the XY model
 * H = -sum_<ij> cos(theta_i - theta_j) (Eq. 5, n=2) on dilute Levy graphs
 * (Eq. 6) with parallel tempering and the E / m
 * observables (Eq. 13-16).  The result is a Markov-chain trajectory, so the
 * oracle is the algorithm step by step in the paper's order; no blocking, fusion or
 * reordering.  fp64 everywhere except where the stored fp32 angle itself is defined
 * (proposal add and wrap, R5), which is fp32 on purpose so that an accepted
 * angle is a well-defined fp32 number.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (see oracle/build_oracle.py).
 *
 * PINS (tests/test_oracle_*.py, all -m "not gpu"):
 *   orc_philox4x32_10      Random123 known-answer vectors (tests/golden/philox4x32_10_kat.txt)
 *   orc_u01                range / symmetry / fp32-exactness
 *   orc_levy_edges         E_b = N z / 2, no duplicates, r_max <= [L/2] sqrt2,
 *                          rho->inf, z=4 gives the square lattice,
 *                          rho=0 gives Poisson(z) degrees, bond-length law
 *   orc_colour_smallest_last  properness bit-exact; 2 colours on the square lattice
 *   orc_measure            dense-matrix numpy evaluation of Eq. 5 / Eq. 16 on small graphs
 *   orc_metropolis_sites   dE == E_total(after) - E_total(before) via orc_measure; beta=0 accepts
 *                          all; rejected move bit-identical; equilibrium vs ring / tree closed
 *                          forms and brute-force quadrature on 3- and 4-site graphs
 *   orc_overrelax_sites    energy conservation, involution, degree-0 no-op, equilibrium pins
 *   orc_pt_swap            acceptance frequency vs min(1,exp(dBeta dE)); inverse permutations;
 *                          PT run reproduces the quadrature values at every temperature
 *   orc_run                all equilibrium pins above run through it
 */
#include "xy_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

static const float ORC_TWO_PI_F = 6.2831855f; /* fp32 nearest to 2 pi (DESIGN R5) */
static const double ORC_TWO_PI = 6.283185307179586476925286766559;

/* ------------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon et al., SC'11): 10 rounds of
 *   (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2;  c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0);
 *   k0 += W0, k1 += W1 after every round.
 * ---------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* DESIGN R11: u = ((x >> 9) + 0.5) * 2^-23, in [2^-24, 1 - 2^-24], exact in fp32. */
float orc_u01(uint32_t x) {
    return ((float)(x >> 9) + 0.5f) * 1.1920928955078125e-07f; /* 2^-23 */
}

/* DESIGN R10: key = (seed_lo, seed_hi); counter = (site, sweep, (sample<<16)|(slot>>1), domain);
 * even slot takes words (x0,x1), odd slot takes (x2,x3). */
void orc_slot_uniforms(uint64_t seed, uint32_t domain, uint32_t site, uint32_t sweep,
                       uint32_t sample, uint32_t slot, float *u1, float *u2) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t ctr[4] = {site, sweep, (sample << 16) | (slot >> 1), domain};
    uint32_t x[4];
    orc_philox4x32_10(ctr, key, x);
    if (slot & 1u) { *u1 = orc_u01(x[2]); *u2 = orc_u01(x[3]); }
    else           { *u1 = orc_u01(x[0]); *u2 = orc_u01(x[1]); }
}

/* ------------------------------------------------------------------------------------------
 * a0. Levy graph (Eq. 6): N z / 2 distinct bonds on the L x L periodic
 * lattice, P(bond ij) proportional to r_ij^-rho with r the minimum-image Euclidean distance.
 * DESIGN R1: site i uniform; partner j != i with P ~ r^-rho over all N-1 displacements
 * d = dy*L + dx, d = 1..N-1.  DESIGN R2: a duplicate {i,j} discards the whole draw.
 * Draw k uses Philox counter (k_lo, k_hi, sample, GRAPH): x0 -> i, (x1, x2) -> 53-bit uniform.
 * Written as the definition: linear scan of the running sum, dense bitmap for duplicates.
 * ---------------------------------------------------------------------------------------- */
static double levy_weight(int L, int d, double rho) {
    int dx = d % L, dy = d / L;
    int mx = dx < L - dx ? dx : L - dx;
    int my = dy < L - dy ? dy : L - dy;
    double r2 = (double)(mx * mx + my * my);
    return pow(r2, -0.5 * rho);
}

int64_t orc_levy_edges(int L, double rho, int z, uint64_t seed, uint32_t sample, int32_t *edges,
                       int64_t max_draws) {
    const int N = L * L;
    const int64_t n_bonds = (int64_t)N * z / 2;
    if (N > 16384 || ((int64_t)N * z) % 2 != 0) return -1;
    uint8_t *present = (uint8_t *)calloc(((size_t)N * N + 7) / 8, 1);
    if (!present) return -1;
    double total = 0.0;
    for (int d = 1; d < N; ++d) total += levy_weight(L, d, rho);
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    int64_t have = 0, k = 0;
    while (have < n_bonds) {
        if (k >= max_draws) { free(present); return -1; }
        uint32_t ctr[4] = {(uint32_t)k, (uint32_t)((uint64_t)k >> 32), sample, ORC_DOMAIN_GRAPH};
        uint32_t x[4];
        orc_philox4x32_10(ctr, key, x);
        ++k;
        int i = (int)(((uint64_t)x[0] * (uint64_t)N) >> 32);
        uint64_t m53 = ((uint64_t)x[1] << 21) | ((uint64_t)x[2] >> 11);
        double v = ((double)m53 + 0.5) * 1.1102230246251565e-16; /* 2^-53 */
        double target = v * total;
        double run = 0.0;
        int d = N - 1;
        for (int dd = 1; dd < N; ++dd) {
            run += levy_weight(L, dd, rho);
            if (run > target) { d = dd; break; }
        }
        int xi = i % L, yi = i / L;
        int xj = (xi + d % L) % L, yj = (yi + d / L) % L;
        int j = yj * L + xj;
        int a = i < j ? i : j, b = i < j ? j : i;
        size_t bit = (size_t)a * N + b;
        if (present[bit >> 3] & (1u << (bit & 7))) continue; /* duplicate: redraw whole bond */
        present[bit >> 3] |= (uint8_t)(1u << (bit & 7));
        edges[2 * have] = i;
        edges[2 * have + 1] = j;
        ++have;
    }
    free(present);
    return k;
}

/* Free boundary conditions ("r up to L sqrt 2"; DESIGN R21), definition level: site i uniform;
 * displacement (dx, dy) in [-(L-1), L-1]^2 without the null vector, P ~ (dx^2 + dy^2)^(-rho/2), by a linear scan of
 * the cumulative sum in index order d = (dy+L-1)(2L-1) + (dx+L-1); partner outside the lattice or duplicate bond:
 * the whole draw is discarded. */
int64_t orc_levy_edges_fbc(int L, double rho, int z, uint64_t seed, uint32_t sample, int32_t *edges,
                           int64_t max_draws) {
    const int N = L * L, W = 2 * L - 1;
    const int64_t n_bonds = (int64_t)N * z / 2;
    if (N > 16384 || ((int64_t)N * z) % 2 != 0) return -1;
    uint8_t *present = (uint8_t *)calloc(((size_t)N * N + 7) / 8, 1);
    if (!present) return -1;
    double total = 0.0;
    for (int d = 0; d < W * W; ++d) {
        const int dx = d % W - (L - 1), dy = d / W - (L - 1);
        if (dx != 0 || dy != 0) total += pow((double)(dx * dx + dy * dy), -0.5 * rho);
    }
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    int64_t have = 0, k = 0;
    while (have < n_bonds) {
        if (k >= max_draws) { free(present); return -1; }
        uint32_t ctr[4] = {(uint32_t)k, (uint32_t)((uint64_t)k >> 32), sample, ORC_DOMAIN_GRAPH};
        uint32_t x[4];
        orc_philox4x32_10(ctr, key, x);
        ++k;
        int i = (int)(((uint64_t)x[0] * (uint64_t)N) >> 32);
        uint64_t m53 = ((uint64_t)x[1] << 21) | ((uint64_t)x[2] >> 11);
        double target = (((double)m53 + 0.5) * 1.1102230246251565e-16) * total;
        double run = 0.0;
        int d = W * W - 1;
        for (int dd = 0; dd < W * W; ++dd) {
            const int dx = dd % W - (L - 1), dy = dd / W - (L - 1);
            if (dx != 0 || dy != 0) run += pow((double)(dx * dx + dy * dy), -0.5 * rho);
            if (run > target) { d = dd; break; }
        }
        int xi = i % L, yi = i / L;
        int xj = xi + d % W - (L - 1), yj = yi + d / W - (L - 1);
        if (xj < 0 || xj >= L || yj < 0 || yj >= L || (xj == xi && yj == yi)) continue;
        int j = yj * L + xj;
        int a = i < j ? i : j, b = i < j ? j : i;
        size_t bit = (size_t)a * N + b;
        if (present[bit >> 3] & (1u << (bit & 7))) continue;
        present[bit >> 3] |= (uint8_t)(1u << (bit & 7));
        edges[2 * have] = i;
        edges[2 * have + 1] = j;
        ++have;
    }
    free(present);
    return k;
}

void orc_csr_from_edges(int N, int n_edges, const int32_t *edges, int32_t *row_ptr,
                        int32_t *col_idx) {
    if (N <= 0) return;
    for (int i = 0; i <= N; ++i) row_ptr[i] = 0;
    for (int e = 0; e < n_edges; ++e) {
        row_ptr[edges[2 * e] + 1]++;
        row_ptr[edges[2 * e + 1] + 1]++;
    }
    for (int i = 0; i < N; ++i) row_ptr[i + 1] += row_ptr[i];
    int32_t *fill = (int32_t *)calloc((size_t)N, sizeof(int32_t));
    for (int e = 0; e < n_edges; ++e) {
        int a = edges[2 * e], b = edges[2 * e + 1];
        col_idx[row_ptr[a] + fill[a]++] = b;
        col_idx[row_ptr[b] + fill[b]++] = a;
    }
    free(fill);
    for (int i = 0; i < N; ++i) { /* insertion sort each row ascending */
        int32_t *row = col_idx + row_ptr[i];
        int n = row_ptr[i + 1] - row_ptr[i];
        for (int p = 1; p < n; ++p) {
            int32_t v = row[p];
            int q = p - 1;
            while (q >= 0 && row[q] > v) { row[q + 1] = row[q]; --q; }
            row[q + 1] = v;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * a1. Colouring: "variant of the Smallest-Last-Ordering".  DESIGN R4:
 * repeatedly remove the vertex of minimum current degree (ties: smallest id); colour in
 * reverse removal order with the smallest colour absent from the coloured neighbours.
 * Written naively, O(N^2).
 * ---------------------------------------------------------------------------------------- */
int orc_colour_smallest_last(int N, const int32_t *row_ptr, const int32_t *col_idx,
                             int32_t *colour) {
    int32_t *deg = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    uint8_t *removed = (uint8_t *)calloc((size_t)N, 1);
    int32_t *order = (int32_t *)malloc((size_t)N * sizeof(int32_t)); /* order[0] removed last */
    for (int v = 0; v < N; ++v) deg[v] = row_ptr[v + 1] - row_ptr[v];
    for (int step = N - 1; step >= 0; --step) {
        int best = -1;
        for (int v = 0; v < N; ++v)
            if (!removed[v] && (best < 0 || deg[v] < deg[best])) best = v;
        order[step] = best;
        removed[best] = 1;
        for (int e = row_ptr[best]; e < row_ptr[best + 1]; ++e)
            if (!removed[col_idx[e]]) deg[col_idx[e]]--;
    }
    for (int v = 0; v < N; ++v) colour[v] = -1;
    int Q = 0;
    for (int step = 0; step < N; ++step) {
        int v = order[step];
        for (int c = 0;; ++c) {
            int used = 0;
            for (int e = row_ptr[v]; e < row_ptr[v + 1]; ++e)
                if (colour[col_idx[e]] == c) { used = 1; break; }
            if (!used) { colour[v] = c; if (c + 1 > Q) Q = c + 1; break; }
        }
    }
    free(deg); free(removed); free(order);
    return Q;
}

/* PAPER.md:490 "sites with a common color are consecutive in the array". */
void orc_renumber_colour_major(int N, const int32_t *row_ptr, const int32_t *col_idx,
                               const int32_t *colour, int32_t *new_to_old, int32_t *row_ptr_new,
                               int32_t *col_idx_new, int32_t *colour_new) {
    int32_t *old_to_new = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int Q = 0;
    for (int v = 0; v < N; ++v) if (colour[v] + 1 > Q) Q = colour[v] + 1;
    int pos = 0;
    for (int c = 0; c < Q; ++c)
        for (int v = 0; v < N; ++v)
            if (colour[v] == c) { new_to_old[pos] = v; old_to_new[v] = pos; ++pos; }
    row_ptr_new[0] = 0;
    for (int a = 0; a < N; ++a) {
        int v = new_to_old[a];
        int n = row_ptr[v + 1] - row_ptr[v];
        int32_t *row = col_idx_new + row_ptr_new[a];
        for (int q = 0; q < n; ++q) row[q] = old_to_new[col_idx[row_ptr[v] + q]];
        for (int p = 1; p < n; ++p) {
            int32_t w = row[p];
            int q = p - 1;
            while (q >= 0 && row[q] > w) { row[q + 1] = row[q]; --q; }
            row[q + 1] = w;
        }
        row_ptr_new[a + 1] = row_ptr_new[a] + n;
        colour_new[a] = colour[v];
    }
    free(old_to_new);
}

int orc_colouring_is_proper(int N, const int32_t *row_ptr, const int32_t *col_idx,
                            const int32_t *colour) {
    for (int i = 0; i < N; ++i)
        for (int e = row_ptr[i]; e < row_ptr[i + 1]; ++e)
            if (colour[i] == colour[col_idx[e]]) return 0;
    return 1;
}

/* ------------------------------------------------------------------------------------------
 * Temperatures.  DESIGN R15: T_k = Tmin (Tmax/Tmin)^(k/(R-1)).  DESIGN R5: beta = fp32(1/T),
 * proposal width w = fp32(2 pi min(1, T/2)) (BASELINE.json config 0).
 * ---------------------------------------------------------------------------------------- */
void orc_geometric_temperatures(int R, double Tmin, double Tmax, double *T) {
    for (int k = 0; k < R; ++k)
        T[k] = (R == 1) ? Tmin : Tmin * pow(Tmax / Tmin, (double)k / (double)(R - 1));
}

void orc_temperature_params(int R, const double *T, float *beta_f, float *w_f) {
    for (int k = 0; k < R; ++k) {
        beta_f[k] = (float)(1.0 / T[k]);
        double half = 0.5 * T[k];
        w_f[k] = (float)(ORC_TWO_PI * (half < 1.0 ? half : 1.0));
    }
}

/* theta = fp32(2 pi_f * u), u from Philox(INIT, sweep 0); uniform in (0, 2 pi). */
void orc_init_theta(int N, int R, uint64_t seed, uint32_t sample, float *theta) {
    for (int i = 0; i < N; ++i)
        for (int r = 0; r < R; ++r) {
            float u1, u2;
            orc_slot_uniforms(seed, ORC_DOMAIN_INIT, (uint32_t)i, 0u, sample, (uint32_t)r, &u1, &u2);
            theta[(size_t)i * R + r] = ORC_TWO_PI_F * u1;
        }
}

/* ------------------------------------------------------------------------------------------
 * a2. Metropolis (PAPER.md:444 "single-spin flip Metropolis update", :454).
 *   proposal  theta' = theta + w (u1 - 1/2)              (BASELINE.json; DESIGN R5; fp32)
 *   dE = - sum_j [cos(theta' - theta_j) - cos(theta - theta_j)]   (Eq. 5, n = 2; fp64)
 *   accept iff u2 < exp(-beta dE)                        (DESIGN R6, strict)
 *   store wrap(theta'): one conditional +-2 pi_f in fp32 (DESIGN R5)
 * ---------------------------------------------------------------------------------------- */
void orc_metropolis_sites(int N, int R, const int32_t *row_ptr, const int32_t *col_idx,
                          float *theta, const int32_t *sites, int n_sites,
                          const float *beta_slot, const float *w_slot, uint64_t seed,
                          uint32_t sweep, uint32_t sample, double *margin, uint8_t *accepted) {
    (void)N;
    for (int k = 0; k < n_sites; ++k) {
        const int i = sites[k];
        for (int r = 0; r < R; ++r) {
            float u1, u2;
            orc_slot_uniforms(seed, ORC_DOMAIN_METROPOLIS, (uint32_t)i, sweep, sample, (uint32_t)r,
                              &u1, &u2);
            const float th = theta[(size_t)i * R + r];
            const float delta = w_slot[r] * (u1 - 0.5f);
            float thp = th + delta;
            double dE = 0.0;
            for (int e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
                const double tj = (double)theta[(size_t)col_idx[e] * R + r];
                dE -= cos((double)thp - tj) - cos((double)th - tj);
            }
            const double p = exp(-(double)beta_slot[r] * dE);
            const int acc = ((double)u2 < p);
            if (margin) margin[(size_t)k * R + r] = fabs((double)u2 - (p < 1.0 ? p : 1.0));
            if (accepted) accepted[(size_t)k * R + r] = (uint8_t)acc;
            if (acc) {
                if (thp >= ORC_TWO_PI_F) thp -= ORC_TWO_PI_F;
                else if (thp < 0.0f) thp += ORC_TWO_PI_F;
                theta[(size_t)i * R + r] = thp;
            }
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * a3. Over-relaxation (ref 66): reflect S_i about the local field
 *   h = sum_j (cos theta_j, sin theta_j);  theta' = 2 atan2(h_y, h_x) - theta  (mod 2 pi).
 * Energy -S_i . h is unchanged.  DESIGN R7: h = 0 exactly (degree 0) leaves theta unchanged.
 * ---------------------------------------------------------------------------------------- */
void orc_overrelax_sites(int N, int R, const int32_t *row_ptr, const int32_t *col_idx,
                         float *theta, const int32_t *sites, int n_sites, double *hnorm) {
    (void)N;
    for (int k = 0; k < n_sites; ++k) {
        const int i = sites[k];
        for (int r = 0; r < R; ++r) {
            double hx = 0.0, hy = 0.0;
            for (int e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
                const double tj = (double)theta[(size_t)col_idx[e] * R + r];
                hx += cos(tj);
                hy += sin(tj);
            }
            if (hnorm) hnorm[(size_t)k * R + r] = sqrt(hx * hx + hy * hy);
            if (hx == 0.0 && hy == 0.0) continue;
            double t = 2.0 * atan2(hy, hx) - (double)theta[(size_t)i * R + r];
            t -= ORC_TWO_PI * floor(t / ORC_TWO_PI);
            float f = (float)t;
            if (f < 0.0f) f = 0.0f;
            theta[(size_t)i * R + r] = f;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * a4. E = -(1/2) sum_i sum_{j in N(i)} cos(theta_i - theta_j)  (Eq. 5 with J in {0,1});
 *     M = sum_i (cos theta_i, sin theta_i)                      (Eq. 16 times N).
 * ---------------------------------------------------------------------------------------- */
void orc_measure(int N, int R, const int32_t *row_ptr, const int32_t *col_idx,
                 const float *theta, double *E, double *Mx, double *My) {
    for (int r = 0; r < R; ++r) {
        double e = 0.0, mx = 0.0, my = 0.0;
        for (int i = 0; i < N; ++i) {
            const double ti = (double)theta[(size_t)i * R + r];
            for (int q = row_ptr[i]; q < row_ptr[i + 1]; ++q)
                e += cos(ti - (double)theta[(size_t)col_idx[q] * R + r]);
            mx += cos(ti);
            my += sin(ti);
        }
        E[r] = -0.5 * e;
        Mx[r] = mx;
        My[r] = my;
    }
}

/* Eq. 13-16: moments of E and m = |M|/N filed under the slot's current temperature. */
void orc_accumulate(int N, int R, const double *E, const double *Mx, const double *My,
                    const int32_t *temp_of_slot, double *acc) {
    for (int r = 0; r < R; ++r) {
        double *a = acc + (size_t)temp_of_slot[r] * ORC_NACC;
        const double mx = Mx[r] / N, my = My[r] / N;
        const double m2 = mx * mx + my * my;
        a[0] += 1.0;
        a[1] += E[r];
        a[2] += E[r] * E[r];
        a[3] += sqrt(m2);
        a[4] += m2;
        a[5] += m2 * m2;
        a[6] += mx;
        a[7] += my;
    }
}

/* ------------------------------------------------------------------------------------------
 * a7. Structure factor at k_min and second-moment correlation length.
 * Eq. 18: C(r) = (1/N) sum_i <S_i . S_{i+r}>; its Fourier transform at momentum k is
 *   chi(k) = (1/N) < |sum_i S_i exp(i k . r_i)|^2 >,  the modulus taken per spin component and added.
 * k_min = (2 pi / L, 0) and (0, 2 pi / L).  chi(0) = N <m^2>.
 * ---------------------------------------------------------------------------------------- */
void orc_fourier(int N, int R, int Lx, int Ly, const int32_t *x, const int32_t *y, const float *theta,
                 double *G1, double *G2) {
    const double two_pi = 6.283185307179586476925286766559;
    for (int r = 0; r < R; ++r) {
        double cre1 = 0, cim1 = 0, sre1 = 0, sim1 = 0, cre2 = 0, cim2 = 0, sre2 = 0, sim2 = 0;
        for (int i = 0; i < N; ++i) {
            const double t = (double)theta[(size_t)i * R + r];
            const double c = cos(t), s = sin(t);
            const double p1 = two_pi * (double)x[i] / (double)Lx, p2 = two_pi * (double)y[i] / (double)Ly;
            cre1 += c * cos(p1); cim1 += c * sin(p1); sre1 += s * cos(p1); sim1 += s * sin(p1);
            cre2 += c * cos(p2); cim2 += c * sin(p2); sre2 += s * cos(p2); sim2 += s * sin(p2);
        }
        G1[r] = (cre1 * cre1 + cim1 * cim1 + sre1 * sre1 + sim1 * sim1) / (double)N;
        G2[r] = (cre2 * cre2 + cim2 * cim2 + sre2 * sre2 + sim2 * sim2) / (double)N;
    }
}

/* Eq. 17: psi = rho - d in the long-range regime, 2 in the short-range regime. */
double orc_xi2(double chi0, double chik, int L, double psi) {
    const double pi = 3.1415926535897932384626433832795;
    return pow(chi0 / chik - 1.0, 1.0 / psi) / (2.0 * sin(pi / (double)L));
}

/* ------------------------------------------------------------------------------------------
 * a8. Random-walk self-return histogram (App. A): "the histogram of return
 * times is proportional to the probability of self-return of a random walker in the graph after a
 * time tau", P(tau) ~ tau^(-dbar/2).  DESIGN R19: every visit of the origin at time tau counts (not
 * only the first return); the simple random walk jumps to a uniformly chosen neighbour.
 * ---------------------------------------------------------------------------------------- */
void orc_random_walk(int N, const int32_t *row_ptr, const int32_t *col_idx, int n_walkers,
                     const int32_t *start, int n_steps, uint64_t seed, uint32_t sample, int64_t *hist) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    (void)N;
    for (int t = 0; t <= n_steps; ++t) hist[t] = 0;
    hist[0] = n_walkers;
    for (int w = 0; w < n_walkers; ++w) {
        int pos = start[w];
        uint32_t x[4] = {0, 0, 0, 0};
        for (int t = 1; t <= n_steps; ++t) {
            const int k = (t - 1) & 3;
            if (k == 0) {
                uint32_t ctr[4] = {(uint32_t)w, (uint32_t)((t - 1) >> 2), sample << 16, ORC_DOMAIN_WALK};
                orc_philox4x32_10(ctr, key, x);
            }
            const int deg = row_ptr[pos + 1] - row_ptr[pos];
            if (deg > 0) pos = col_idx[row_ptr[pos] + (int)(((uint64_t)x[k] * (uint64_t)deg) >> 32)];
            if (pos == start[w]) hist[t] += 1;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * a5. Parallel tempering (ref 65).  DESIGN R9: round k attempts the pairs
 * (t, t+1) with t = k mod 2, k mod 2 + 2, ...;  a = slot_of_temp[t], b = slot_of_temp[t+1];
 *   accept iff u < exp((beta_t - beta_{t+1}) (E_a - E_b)),   beta = 1/T in fp64;
 * on accept the two temperature LABELS are exchanged, spins stay where they are.
 * u = u01(x0) of Philox counter (t, round, sample<<16, SWAP).
 * ---------------------------------------------------------------------------------------- */
void orc_pt_swap(int R, const double *T, const double *E_slot, int32_t *slot_of_temp,
                 int32_t *temp_of_slot, uint64_t seed, uint32_t round, uint32_t sample,
                 const uint8_t *decisions_in, uint8_t *decisions_out, double *margin_out) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    for (int t = (int)(round & 1u); t + 1 < R; t += 2) {
        const int a = slot_of_temp[t], b = slot_of_temp[t + 1];
        uint32_t ctr[4] = {(uint32_t)t, round, sample << 16, ORC_DOMAIN_SWAP};
        uint32_t x[4];
        orc_philox4x32_10(ctr, key, x);
        const double u = (double)orc_u01(x[0]);
        const double arg = (1.0 / T[t] - 1.0 / T[t + 1]) * (E_slot[a] - E_slot[b]);
        const double p = exp(arg);
        int acc = decisions_in ? (int)decisions_in[t] : (u < p);
        if (decisions_out) decisions_out[t] = (uint8_t)acc;
        if (margin_out) margin_out[t] = fabs(u - (p < 1.0 ? p : 1.0));
        if (acc) {
            slot_of_temp[t] = b;
            slot_of_temp[t + 1] = a;
            temp_of_slot[a] = t + 1;
            temp_of_slot[b] = t;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * a6. The protocol (BASELINE.json config 0: 1 OR sweep per Metropolis sweep,
 * swaps every `sweeps_per_swap` sweeps).  Colours are processed sequentially, same-colour sites
 * are mutually independent.
 * ---------------------------------------------------------------------------------------- */
void orc_run_order(int N, int R, int Q, const int32_t *row_ptr, const int32_t *col_idx,
                   const int32_t *class_ptr, float *theta, const double *T, int32_t *temp_of_slot,
                   int32_t *slot_of_temp, uint64_t seed, uint32_t sample, uint32_t *sweep,
                   uint32_t *round, int n_cycles, int sweeps_per_swap, int or_per_sweep,
                   int measure_every, int order, double *acc, int64_t *swap_attempts,
                   int64_t *swap_accepts) {
    float *beta_f = (float *)malloc((size_t)R * sizeof(float));
    float *w_f = (float *)malloc((size_t)R * sizeof(float));
    float *beta_slot = (float *)malloc((size_t)R * sizeof(float));
    float *w_slot = (float *)malloc((size_t)R * sizeof(float));
    double *E = (double *)malloc((size_t)R * sizeof(double));
    double *Mx = (double *)malloc((size_t)R * sizeof(double));
    double *My = (double *)malloc((size_t)R * sizeof(double));
    int32_t *sites = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    uint8_t *dec = (uint8_t *)calloc((size_t)R, 1);
    for (int i = 0; i < N; ++i) sites[i] = i;
    orc_temperature_params(R, T, beta_f, w_f);

    for (int cycle = 0; cycle < n_cycles; ++cycle) {
        for (int r = 0; r < R; ++r) {
            beta_slot[r] = beta_f[temp_of_slot[r]];
            w_slot[r] = w_f[temp_of_slot[r]];
        }
        for (int k = 0; k < sweeps_per_swap; ++k) {
            *sweep += 1u;
            if (order == 1) {
                /* interleaved order: per colour class, Metropolis and then the
                 * over-relaxation of its sites; every update leaves the Gibbs measure invariant, so
                 * any fixed order of the same updates is a valid chain. */
                for (int c = 0; c < Q; ++c) {
                    orc_metropolis_sites(N, R, row_ptr, col_idx, theta, sites + class_ptr[c],
                                         class_ptr[c + 1] - class_ptr[c], beta_slot, w_slot, seed,
                                         *sweep, sample, NULL, NULL);
                    orc_overrelax_sites(N, R, row_ptr, col_idx, theta, sites + class_ptr[c],
                                        class_ptr[c + 1] - class_ptr[c], NULL);
                }
            } else {
                for (int c = 0; c < Q; ++c)
                    orc_metropolis_sites(N, R, row_ptr, col_idx, theta, sites + class_ptr[c],
                                         class_ptr[c + 1] - class_ptr[c], beta_slot, w_slot, seed,
                                         *sweep, sample, NULL, NULL);
                for (int o = 0; o < or_per_sweep; ++o)
                    for (int c = 0; c < Q; ++c)
                        orc_overrelax_sites(N, R, row_ptr, col_idx, theta, sites + class_ptr[c],
                                            class_ptr[c + 1] - class_ptr[c], NULL);
            }
            if (measure_every > 0 && (*sweep % (uint32_t)measure_every) == 0u) {
                orc_measure(N, R, row_ptr, col_idx, theta, E, Mx, My);
                orc_accumulate(N, R, E, Mx, My, temp_of_slot, acc);
            }
        }
        orc_measure(N, R, row_ptr, col_idx, theta, E, Mx, My);
        orc_pt_swap(R, T, E, slot_of_temp, temp_of_slot, seed, *round, sample, NULL, dec, NULL);
        for (int t = (int)(*round & 1u); t + 1 < R; t += 2) {
            if (swap_attempts) swap_attempts[t] += 1;
            if (swap_accepts) swap_accepts[t] += dec[t];
        }
        *round += 1u;
    }
    free(beta_f); free(w_f); free(beta_slot); free(w_slot);
    free(E); free(Mx); free(My); free(sites); free(dec);
}

void orc_run(int N, int R, int Q, const int32_t *row_ptr, const int32_t *col_idx,
             const int32_t *class_ptr, float *theta, const double *T, int32_t *temp_of_slot,
             int32_t *slot_of_temp, uint64_t seed, uint32_t sample, uint32_t *sweep,
             uint32_t *round, int n_cycles, int sweeps_per_swap, int or_per_sweep,
             int measure_every, double *acc, int64_t *swap_attempts, int64_t *swap_accepts) {
    orc_run_order(N, R, Q, row_ptr, col_idx, class_ptr, theta, T, temp_of_slot, slot_of_temp, seed,
                  sample, sweep, round, n_cycles, sweeps_per_swap, or_per_sweep, measure_every, 0, acc,
                  swap_attempts, swap_accepts);
}
