/*
 * xy_oracle.h -- CPU ORACLE for the XY-on-Levy-graph hot path of arXiv 1211.3991.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code
 * with the CUDA path (own Philox, own CSR walk, own reductions) and neither side
 * includes the other.
 *
 * Plain single-threaded C, fp64 for every energy / acceptance / reduction; angles are
 * stored as fp32 because the paper stores them so (App. B.c, "single
 * precision (4 bytes) for the storing of floating-point numbers", :494).
 *
 * Each function cites the passage it follows (PAPER.md line, section) or the reading
 * listed in DESIGN.md section 3 ("Readings").  What pins each function is listed in
 * DESIGN.md section 4 and in the header comment of xy_oracle.c.
 */
#ifndef XY_ORACLE_H
#define XY_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Philox domains (reading R10). */
#define ORC_DOMAIN_INIT 0u
#define ORC_DOMAIN_METROPOLIS 1u
#define ORC_DOMAIN_SWAP 2u
#define ORC_DOMAIN_GRAPH 3u
#define ORC_DOMAIN_WALK 4u

/* accumulator columns per (temperature) */
#define ORC_NACC 8 /* n, E, E^2, |m|, m^2, m^4, Mx/N, My/N */

/* ---- counter-based RNG (BASELINE.json north_star: Philox4x32-10) ---- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
float orc_u01(uint32_t x);
/* the two uniforms (u1 proposal, u2 acceptance) of (site, sweep, sample, slot) in `domain` */
void orc_slot_uniforms(uint64_t seed, uint32_t domain, uint32_t site, uint32_t sweep,
                       uint32_t sample, uint32_t slot, float *u1, float *u2);

/* ---- a0: Levy graph, definition level (Eq. 6; DESIGN R1,R2) ---- */
/* returns number of Philox draws consumed (>=E_b) or -1 on failure; edges[2*e], edges[2*e+1] */
int64_t orc_levy_edges(int L, double rho, int z, uint64_t seed, uint32_t sample,
                       int32_t *edges /*[N*z/2][2]*/, int64_t max_draws);
/* free boundary conditions (DESIGN R21): plain Euclidean distance on the open lattice */
int64_t orc_levy_edges_fbc(int L, double rho, int z, uint64_t seed, uint32_t sample,
                           int32_t *edges /*[N*z/2][2]*/, int64_t max_draws);
/* symmetric CSR with ascending neighbour lists from an edge list */
void orc_csr_from_edges(int N, int n_edges, const int32_t *edges, int32_t *row_ptr /*[N+1]*/,
                        int32_t *col_idx /*[2*n_edges]*/);

/* ---- a1: smallest-last greedy colouring (App. B.a; DESIGN R4) ---- */
/* returns Q; colour[v] in [0,Q) */
int orc_colour_smallest_last(int N, const int32_t *row_ptr, const int32_t *col_idx,
                             int32_t *colour /*[N]*/);
/* colour-major renumbering: new_to_old sorted by (colour, old id); outputs renumbered CSR+colour */
void orc_renumber_colour_major(int N, const int32_t *row_ptr, const int32_t *col_idx,
                               const int32_t *colour, int32_t *new_to_old /*[N]*/,
                               int32_t *row_ptr_new /*[N+1]*/, int32_t *col_idx_new,
                               int32_t *colour_new /*[N]*/);
/* 1 iff no edge joins equal colours */
int orc_colouring_is_proper(int N, const int32_t *row_ptr, const int32_t *col_idx,
                            const int32_t *colour);

/* ---- temperatures and per-slot parameters (DESIGN R5, R15) ---- */
void orc_geometric_temperatures(int R, double Tmin, double Tmax, double *T /*[R]*/);
void orc_temperature_params(int R, const double *T, float *beta_f /*[R]*/, float *w_f /*[R]*/);

/* ---- state init (DESIGN R10: domain INIT) ---- */
void orc_init_theta(int N, int R, uint64_t seed, uint32_t sample, float *theta /*[N][R]*/);

/* ---- a2: Metropolis single-spin update of a list of mutually non-adjacent sites
 *      (App. B; proposal BASELINE.json config 0; DESIGN R5,R6) ----
 * theta [N][R] updated in place.  beta_slot/w_slot are per memory slot (lane).
 * margin[k*R+r] (may be NULL) = |u2 - min(1, exp(-beta dE))| for list entry k;
 * accepted[k*R+r] (may be NULL) = 1 iff the move was accepted. */
void orc_metropolis_sites(int N, int R, const int32_t *row_ptr, const int32_t *col_idx,
                          float *theta, const int32_t *sites, int n_sites,
                          const float *beta_slot, const float *w_slot, uint64_t seed,
                          uint32_t sweep, uint32_t sample, double *margin, uint8_t *accepted);

/* ---- a3: over-relaxation (App. B.b, ref 66; DESIGN R7) ----
 * hnorm[k*R+r] (may be NULL) = |h| of the local field for list entry k. */
void orc_overrelax_sites(int N, int R, const int32_t *row_ptr, const int32_t *col_idx,
                         float *theta, const int32_t *sites, int n_sites, double *hnorm);

/* ---- a4: observables of one configuration (PAPER.md:90-94 Eq. 5; :179-181 Eq. 16) ---- */
void orc_measure(int N, int R, const int32_t *row_ptr, const int32_t *col_idx,
                 const float *theta, double *E /*[R]*/, double *Mx /*[R]*/, double *My /*[R]*/);
/* file one measurement under each slot's current temperature (Eq. 13-16) */
void orc_accumulate(int N, int R, const double *E, const double *Mx, const double *My,
                    const int32_t *temp_of_slot, double *acc /*[R][ORC_NACC]*/);

/* ---- a7: structure factor at the smallest momenta and the second-moment correlation
 *      length (Eq. 17-18) ----
 * G1[r] = |sum_i S_i exp(i 2 pi x_i / Lx)|^2 / N, G2[r] likewise with y_i / Ly, S_i = (cos th_i, sin th_i): the
 * single-configuration estimators of chi(k_min) for k_min = (2 pi / L, 0) and (0, 2 pi / L); chi(0) = N m^2. */
void orc_fourier(int N, int R, int Lx, int Ly, const int32_t *x /*[N]*/, const int32_t *y /*[N]*/,
                 const float *theta /*[N][R]*/, double *G1 /*[R]*/, double *G2 /*[R]*/);
/* Eq. 17: xi_2 = [chi(0)/chi(k_min) - 1]^(1/psi) / (2 sin(pi / L)) */
double orc_xi2(double chi0, double chik, int L, double psi);

/* ---- a8: random-walk self-return histogram for the spectral dimension
 *      (Eq. 11 P(tau) ~ tau^(-dbar/2); :436-440 App. A; DESIGN R19) ----
 * Walker w starts at start[w]; at step t = 1..n_steps it moves to a uniformly chosen neighbour of its site
 * (stays if the site has none); hist[t] += 1 whenever it is back at start[w] after step t (hist[0] = n_walkers).
 * Neighbour k = (x * deg) >> 32 with x = word (t-1) % 4 of Philox counter (w, (t-1)/4, sample << 16, WALK). */
void orc_random_walk(int N, const int32_t *row_ptr, const int32_t *col_idx, int n_walkers,
                     const int32_t *start, int n_steps, uint64_t seed, uint32_t sample,
                     int64_t *hist /*[n_steps+1]*/);

/* ---- a5: one parallel-tempering swap round (App. B.b, ref 65; DESIGN R9) ----
 * decisions_in NULL: draw u from Philox(SWAP) and decide; else use decisions_in[t] for pair (t,t+1).
 * decisions_out[t], margin_out[t] (may be NULL) are written for every attempted pair. */
void orc_pt_swap(int R, const double *T, const double *E_slot, int32_t *slot_of_temp,
                 int32_t *temp_of_slot, uint64_t seed, uint32_t round, uint32_t sample,
                 const uint8_t *decisions_in, uint8_t *decisions_out, double *margin_out);

/* ---- a6: the whole protocol on one sample (DESIGN section 2 "order binds both paths") ----
 * state in/out: theta, temp_of_slot, slot_of_temp, *sweep, *round; acc += measurements.
 * class_ptr[Q+1] delimits colour classes of the colour-major numbering.
 * swap_attempts/swap_accepts [R-1] (may be NULL) are incremented per pair. */
void orc_run(int N, int R, int Q, const int32_t *row_ptr, const int32_t *col_idx,
             const int32_t *class_ptr, float *theta, const double *T, int32_t *temp_of_slot,
             int32_t *slot_of_temp, uint64_t seed, uint32_t sample, uint32_t *sweep,
             uint32_t *round, int n_cycles, int sweeps_per_swap, int or_per_sweep,
             int measure_every, double *acc /*[R][ORC_NACC]*/, int64_t *swap_attempts,
             int64_t *swap_accepts);

/* the same with the order of a sweep as a parameter: 0 = as orc_run, 1 = interleaved by colour (per colour
 * class: Metropolis, then over-relaxation of its sites; needs or_per_sweep == 1) */
void orc_run_order(int N, int R, int Q, const int32_t *row_ptr, const int32_t *col_idx,
                   const int32_t *class_ptr, float *theta, const double *T, int32_t *temp_of_slot,
                   int32_t *slot_of_temp, uint64_t seed, uint32_t sample, uint32_t *sweep,
                   uint32_t *round, int n_cycles, int sweeps_per_swap, int or_per_sweep,
                   int measure_every, int order, double *acc, int64_t *swap_attempts,
                   int64_t *swap_accepts);

#ifdef __cplusplus
}
#endif
#endif
