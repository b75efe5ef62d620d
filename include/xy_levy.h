/*
 * xy_levy.h -- host-side Levy-graph builder and greedy colouring (C ABI, no CUDA).
 *
 * This is the SEEDED INPUT GENERATOR shared by the CUDA path's harness and by the tests that
 * drive the oracle (BASELINE.json north_star, subsystem (1)).  It
 * holds none of the Monte-Carlo arithmetic.  oracle/xy_oracle.c carries an independent,
 * definition-level restatement (orc_levy_edges, orc_colour_smallest_last) against which the
 * output of this library is checked bit-exactly in tests/test_builder.py.
 *
 * a0 (Eq. 6): N z / 2 distinct bonds on the L x L periodic lattice,
 *    P(bond ij) ~ r_ij^-rho, r the minimum-image Euclidean distance (r_max = [L/2] sqrt 2).
 *    Reading R1/R2: draw k = 0,1,2,... takes Philox4x32-10 counter
 *    (k_lo, k_hi, sample, 3), key (seed_lo, seed_hi);  i = (x0 * N) >> 32;
 *    v = (((x1 << 21) | (x2 >> 11)) + 0.5) 2^-53;  displacement d = dy L + dx in [1, N-1] is the
 *    first index whose running sum of w_d = (r_d^2)^(-rho/2) (summed in index order, fp64)
 *    exceeds v * total;  j = ((y_i+dy) mod L) L + (x_i+dx) mod L;  a bond already present
 *    discards the draw.
 * a1 (App. B.a): smallest-last ordering (remove the vertex of minimum current
 *    degree, ties to the smallest id), greedy smallest-free colour in reverse removal order.
 *    Then sites are renumbered colour-major ("sites with a common color are
 *    consecutive in the array"), old (lattice) order kept inside a class; neighbour lists are
 *    ascending in the new numbering.
 *
 * All arrays are HOST memory owned by the caller.  Return 0 on success, negative on error
 * (XY_LEVY_EINVAL bad argument, XY_LEVY_ENOMEM, XY_LEVY_EDRAWS draw limit hit); the message is
 * in xy_levy_last_error() (thread-local).  No exceptions, no aborts.
 */
#ifndef XY_LEVY_H
#define XY_LEVY_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define XY_LEVY_OK 0
#define XY_LEVY_EINVAL (-1)
#define XY_LEVY_ENOMEM (-2)
#define XY_LEVY_EDRAWS (-3)

/* Build S samples (global sample ids sample_base .. sample_base+S-1), colour and renumber them.
 *   row_ptr    [S][N+1]   CSR row pointers, nnz = N*z for every sample
 *   col_idx    [S][N*z]   neighbour ids (new numbering), ascending per row
 *   colour     [S][N]     colour of each (new) site id, non-decreasing in the id
 *   new_to_old [S][N]     lattice id y*L+x of each new site id        (may be NULL)
 *   n_colours  [S]        Q per sample                                 (may be NULL)
 *   n_draws    [S]        Philox draws consumed per sample             (may be NULL)
 * n_threads <= 0 picks the hardware concurrency; samples are built independently. */
int xy_levy_build(int L, double rho, int z, uint64_t seed, uint32_t sample_base, int S,
                  int n_threads, int32_t *row_ptr, int32_t *col_idx, int32_t *colour,
                  int32_t *new_to_old, int32_t *n_colours, int64_t *n_draws);

/* The same with FREE boundary conditions (Fig. 14: bond lengths up to L sqrt 2 instead of
 * [L/2] sqrt 2): plain Euclidean distance on the open L x L lattice.  A bond is drawn by choosing i uniformly and a
 * displacement (dx, dy) in [-(L-1), L-1]^2 \ {0} with P ~ |d|^-rho (one fp64 CDF summed in index order
 * d = (dy+L-1)(2L-1) + (dx+L-1)); a partner outside the lattice or a duplicate bond discards the whole draw, so the
 * accepted bonds are distributed ~ r_ij^-rho over the pairs that exist (DESIGN R21).  L <= 2048. */
int xy_levy_build_fbc(int L, double rho, int z, uint64_t seed, uint32_t sample_base, int S,
                  int n_threads, int32_t *row_ptr, int32_t *col_idx, int32_t *colour,
                  int32_t *new_to_old, int32_t *n_colours, int64_t *n_draws);

/* xy_levy_build / xy_levy_build_fbc with one more step between the colouring and the renumbering: if
 * reduce_moves_per_site > 0 the smallest-last colouring is passed through xy_colour_reduce (max_moves =
 * reduce_moves_per_site * N, key = seed, sample = the global sample id) until it stops losing colours.  On the z = 6
 * Levy graphs this keeps Q = 5 (they contain 5-cliques) but shrinks the fifth class from ~1.4 % of the sites to a few
 * dozen, and evens out the other four.  The bonds are the same as without the step; only the colours -- and with them
 * the site numbering -- differ.  free_boundaries != 0 selects the free-boundary construction. */
int xy_levy_build_opt(int free_boundaries, int reduce_moves_per_site, int L, double rho, int z, uint64_t seed,
                      uint32_t sample_base, int S, int n_threads, int32_t *row_ptr, int32_t *col_idx, int32_t *colour,
                      int32_t *new_to_old, int32_t *n_colours, int64_t *n_draws);

/* Smallest-last greedy colouring of any symmetric CSR graph; returns Q (>= 0) or a negative error. */
int xy_colour_smallest_last(int N, const int32_t *row_ptr, const int32_t *col_idx,
                            int32_t *colour /*[N]*/);

/* Fewer colours, or a smaller last colour class, by local search (any proper colouring is a correct
 * result; PAPER.md:456 reports Q, :494 time ~ Q/2).  colour[] (in/out) must be a proper colouring with colours 0..Q-1.
 * While Q > target_q: the sites of the last class are given the least conflicting of the other colours and a tabu /
 * min-conflicts search (conflicting site chosen by Philox4x32-10 counter (move_lo, move_hi, sample, 5), key = seed; it
 * takes its least conflicting non-tabu colour) repairs the monochromatic bonds.  If max_moves moves do not repair all of
 * them (a graph with a Q-clique cannot lose its Q-th colour), conflicting sites without a free colour may go back to
 * the last colour (never two neighbours): same Q, but a last class of a few sites instead of ~1.4 % of them.
 * Deterministic.  Returns the final number of colours (>= target_q) or a negative error.  The result
 * is always proper (tests/test_builder.py checks it with the oracle's checker). */
int xy_colour_reduce(int N, const int32_t *row_ptr, const int32_t *col_idx, int32_t *colour /*[N] in/out*/, int target_q,
                     uint64_t seed, uint32_t sample, int64_t max_moves);

/* Colour-major renumbering of any coloured CSR graph (same outputs as the per-sample arrays above). */
int xy_renumber_colour_major(int N, const int32_t *row_ptr, const int32_t *col_idx,
                             const int32_t *colour, int32_t *new_to_old, int32_t *row_ptr_new,
                             int32_t *col_idx_new, int32_t *colour_new);

const char *xy_levy_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
