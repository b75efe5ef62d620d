/*
 * xy_b200.h -- C ABI of the B200 (sm_100a) hot path of arXiv 1211.3991:
 * graph-coloured Metropolis + over-relaxation sweeps of the XY model
 *     H = - sum_<ij> cos(theta_i - theta_j)                      (Eq. 5, n = 2)
 * on S independent graph samples (Eq. 12) x R parallel-tempering replicas
 * (PAPER.md:460-472), with per-sweep E / m reductions (Eq. 13-16) and on-device
 * temperature-label swaps.  Every step runs in hand-written CUDA kernels; there is no CPU fallback:
 * without a CUDA device every call that touches the device returns XY_ECUDA.
 *
 * Conventions
 *   - every function returns int: XY_OK (0) or a negative code; the message of the last failure on the
 *     calling thread is xy_last_error().  No exceptions, no aborts.
 *   - "host" pointers are borrowed for the duration of the call and copied; "device" pointers must stay
 *     valid while the handle lives.  Handles are owned by the library (xy_graph_free / xy_pt_destroy).
 *   - `stream` is a cudaStream_t passed as void* (e.g. torch.cuda.current_stream().cuda_stream);
 *     xy_pt_create(stream = NULL) makes the library create a private non-blocking stream (CUDA graphs
 *     cannot be captured on the legacy default stream).  All work of a handle is enqueued on its stream;
 *     calls return without synchronising unless they hand data back to the host.
 *   - layouts: theta[S][N][R] fp32 radians in [0, 2pi_f], replica (memory slot) fastest
 *     (BASELINE.json north_star); labels temp_of_slot[S][R], slot_of_temp[S][R] int32, mutually inverse;
 *     "slot" = memory lane of a replica, "temperature" = index into T[]; swaps move labels, not spins.
 *   - site numbering must be COLOUR-MAJOR: colour[] non-decreasing in the site id (PAPER.md:490
 *     "sites with a common color are consecutive in the array"); xy_renumber_colour_major() in
 *     xy_levy.h produces it for any coloured graph.
 *   - random numbers: Philox4x32-10, key = (seed_lo, seed_hi),
 *     counter = (site, sweep, (global_sample << 16) | (slot >> 1), domain); even slot takes (x0, x1),
 *     odd slot (x2, x3); u = ((x >> 9) + 0.5) 2^-23.  domain 0 = init, 1 = Metropolis, 2 = swap
 *     (site = t, sweep = round, slot = 0).  global_sample = sample_base + s < 65536, R <= 131072.
 *   - order of one PT cycle (binds this library and the oracle):
 *       repeat sweeps_per_swap times: sweep += 1; Metropolis colours 0..Q-1; or_per_sweep x (OR colours
 *       0..Q-1); measure+accumulate iff sweep % measure_every == 0;   then one swap round; round += 1.
 */
#ifndef XY_B200_H
#define XY_B200_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define XY_OK 0
#define XY_EINVAL (-1) /* bad argument */
#define XY_ENOMEM (-2) /* host or device allocation failed */
#define XY_ECUDA (-3)  /* CUDA runtime error, or no CUDA device */
#define XY_EGRAPH (-4) /* malformed graph or improper colouring */
#define XY_ESTATE (-5) /* call not valid in the handle's current state */

#define XY_NACC 8 /* accumulator columns: n, E, E^2, |m|, m^2, m^4, Mx/N, My/N */

typedef struct xy_graph xy_graph;
typedef struct xy_pt xy_pt;

const char *xy_last_error(void);
/* ABI version of this header (bumped on any signature change). */
int xy_abi_version(void);

/* ---- graph (SURVEY.md 8(b); PAPER.md:94 J_ij in {0,1}; :452-456 colouring; :490 adjacency list) ----
 * S samples of N sites each.  row_ptr [S][N+1] (each sample starts at 0), col_idx = the S neighbour
 * arrays concatenated (sample s has row_ptr[s][N] entries, site ids local to the sample), colour [S][N].
 * Validated per sample: row_ptr monotone from 0; ids in range; no self-loop; no duplicate; symmetric;
 * colour >= 0 and non-decreasing in the site id; NO MONOCHROMATIC EDGE.  Any violation -> XY_EGRAPH.
 * Degree-0 sites, trees, rings, 2-site graphs are all fine.  Copies everything to the device. */
int xy_graph_load(int S, int N, const int32_t *row_ptr /*host*/, const int32_t *col_idx /*host*/,
                  const int32_t *colour /*host*/, void *stream, xy_graph **out);
int xy_graph_free(xy_graph *g);
/* any output pointer may be NULL */
int xy_graph_info(const xy_graph *g, int *S, int *N, int64_t *nnz_total, int *q_max, int *max_degree);

/* Lattice coordinates of the sites (needed only by xy_measure_fourier): x, y [S][N] host, 0 <= x < Lx, 0 <= y < Ly,
 * Lx, Ly <= 65535.  For a Levy graph built by xy_levy_build: x = new_to_old % L, y = new_to_old / L.  Synchronous. */
int xy_graph_set_coords(xy_graph *g, int Lx, int Ly, const int32_t *x /*host*/, const int32_t *y /*host*/);

/* Random-walk self-return histogram on the loaded graphs, for the spectral dimension (Eq. 11
 * P(tau) ~ tau^(-dbar/2); :436-440 App. A).  For every sample, walker w starts at
 * start[s][w] (host, [S][n_walkers]) and makes n_steps (<= 12000) jumps to a uniformly chosen neighbour (it stays on a
 * site without neighbours); hist_host [S][n_steps+1] (host, int64) counts, per time t, the walkers that are back at
 * their origin after step t (every visit counts; hist[s][0] = n_walkers).  Neighbour choice: (x * degree) >> 32 with
 * x = word (t-1) % 4 of Philox4x32-10 counter (w, (t-1)/4, (sample_base + s) << 16, 4), key = seed.  Integer work,
 * bit-exact against the oracle.  Runs on `stream` (cudaStream_t as void*, NULL = default) and synchronises it. */
int xy_random_walk(const xy_graph *g, int n_walkers, const int32_t *start /*host*/, int n_steps, uint64_t seed,
                   uint32_t sample_base, void *stream, int64_t *hist_host);

/* xy_random_walk for callers that cannot allocate: the SAME kernel and the same results, but this entry point calls no
 * cudaMalloc / cudaFree (nor any other allocating CUDA routine).  start_dev [S][n_walkers] int32 and hist_dev
 * [S][n_steps+1] int64 are DEVICE buffers of the caller (on the graph's device); the 64-bit histogram the kernel's atomics
 * accumulate into -- the buffer xy_random_walk allocates per call -- is a file-scope static __device__ array of
 * XY_WALK_STATIC_ENTRIES (65536) 64-bit words = 512 KiB, which every GPU that loads the library holds until exit; its
 * address is taken once per device with cudaGetSymbolAddress.  XY_EINVAL if S * (n_steps + 1) > XY_WALK_STATIC_ENTRIES
 * (or a start site is out of range: the start sites are checked on the device).  The call clears the words it uses,
 * runs the walk, copies them to hist_dev and synchronises `stream`.  ALL calls on a device share the one array, which
 * keeps the last call's contents: calls that overlap on the GPU (two streams, two host threads) race -- serialise them. */
#define XY_WALK_STATIC_ENTRIES 65536
int xy_random_walk_static(const xy_graph *g, int n_walkers, const int32_t *start_dev /*device*/, int n_steps, uint64_t seed,
                          uint32_t sample_base, void *stream, int64_t *hist_dev /*device*/);

/* Device time in microseconds of the k_random_walk launch of the calling thread's last successful xy_random_walk call
 * (CUDA events around the kernel alone, on that call's stream: no allocation, no copy).  XY_ESTATE if there was none. */
int xy_random_walk_kernel_us(double *us_out);

/* ---- PT ensemble ----
 * T [R] host, strictly positive, ascending (T = +inf allowed: beta = 0).  width [R] host or NULL;
 * NULL selects the BASELINE.json proposal width 2 pi min(1, T/2).  beta and width are rounded to fp32
 * per temperature for the Metropolis kernel; the swap rule uses 1/T in fp64.
 * theta_dev: device buffer [S][N][R] fp32 owned by the caller (8-byte aligned), or NULL to let the
 * library allocate.  Initialises theta = 2pi_f * u (Philox domain 0), identity labels, counters 0,
 * accumulators 0.  The graph must outlive the ensemble. */
int xy_pt_create(const xy_graph *g, int R, const double *T /*host*/, const double *width /*host|NULL*/,
                 uint64_t seed, uint32_t sample_base, float *theta_dev /*device|NULL*/, void *stream,
                 xy_pt **out);
int xy_pt_destroy(xy_pt *pt);

/* ---- the hot-path calls named by BASELINE.json north_star ---- */
/* n Metropolis sweeps: colours 0..Q-1 in order, sweep counter += 1 per sweep. */
int xy_sweep(xy_pt *pt, int n_sweeps);
/* One Metropolis sweep exactly as xy_sweep(pt, 1), which also reports the ACCEPTANCE RATE of the proposals per temperature
 * (SURVEY.md section 5 metrics; the rate the proposal width 2 pi min(1, T/2) of BASELINE.json is meant to keep usable):
 * acc_host[s][t] (host, [S][R] doubles, indexed by temperature) = sites of sample s whose angle in the slot of
 * temperature t changed / N.  An accepted proposal always changes the stored angle except when |delta| is below half an
 * ulp of the angle (probability ~1e-7 per update).  Costs one device copy of theta (scratch memory of theta's size,
 * freed before returning) and one comparison pass; synchronises the stream. */
int xy_sweep_acceptance(xy_pt *pt, double *acc_host);
/* n over-relaxation sweeps (ref 66): no randoms, counters untouched. */
int xy_overrelax(xy_pt *pt, int n_sweeps);
/* one swap round (ref 65): pairs (t,t+1), t = round mod 2 (mod 2); energies are
 * recomputed first unless still fresh; accept iff u < exp((beta_t-beta_t+1)(E_a-E_b)); round += 1. */
int xy_pt_swap(xy_pt *pt);
/* E, M_x, M_y of every replica (Eq. 5, Eq. 16), added to the fp64 accumulators of the replica's
 * current temperature (Eq. 13-15).  out_host: [S][R][3] doubles (E, Mx, My) indexed by TEMPERATURE,
 * or NULL; a non-NULL out_host synchronises the stream. */
int xy_measure(xy_pt *pt, double *out_host);

/* Structure factor at the smallest momenta (Eq. 17-18): for every replica
 * G1 = |sum_i S_i exp(i 2 pi x_i / Lx)|^2 / N and G2 likewise with y_i / Ly -- the single-configuration estimators of
 * chi(k_min), k_min = (2 pi / L, 0) and (0, 2 pi / L); added to the fp64 accumulators (n, sum G1, sum G2) of the
 * replica's current temperature (xy_read_fourier_accumulators; cleared by xy_reset_accumulators).  chi(0) = N <m^2>
 * comes from the ordinary accumulators, xi_2 = [chi(0)/chi(k_min) - 1]^(1/psi) / (2 sin(pi / L)).
 * out_host: [S][R][2] doubles (G1, G2) indexed by TEMPERATURE, or NULL; non-NULL synchronises the stream.
 * XY_ESTATE unless xy_graph_set_coords has been called. */
int xy_measure_fourier(xy_pt *pt, double *out_host);
int xy_read_fourier_accumulators(xy_pt *pt, double *acc_host /*[S][R][3]: n, sum G1, sum G2 by temperature*/);

/* n_cycles PT cycles in the order stated at the top, replayed from a captured CUDA graph (SURVEY.md
 * 8(a) row a6).  measure_every = 0 disables measurements (energies are still computed for the swap).
 * sweeps_per_swap >= 1, or_per_sweep >= 0. */
int xy_run(xy_pt *pt, int n_cycles, int sweeps_per_swap, int or_per_sweep, int measure_every);

/* n_blocks x [ sweeps_per_block x (one Metropolis sweep + or_per_sweep OR sweeps) ], no measurement and no
 * swap, in the same group schedule and from the same kind of captured graph as xy_run: the bare coloured
 * Metropolis + over-relaxation sweep of SURVEY.md 8(d) "(A)".  sweep counter += n_blocks*sweeps_per_block. */
int xy_run_sweeps(xy_pt *pt, int n_blocks, int sweeps_per_block, int or_per_sweep);

/* Samples are independent, so a cycle may be executed for groups of `samples_per_group` samples at a
 * time (all sweeps of the cycle for group 0, then group 1, ...) to keep a group L2-resident; results
 * are bit-identical for every value.  0 = automatic (default), S = all samples per launch. */
int xy_set_schedule(xy_pt *pt, int samples_per_group);

/* Execution path of xy_run / xy_run_sweeps ("subsets ... processed sequentially on
 * each MCS").  1 = one launch per colour class (k_phase) captured in a CUDA graph with programmatic-dependent-launch
 * edges: right when a class fills the chip.  2 = one THREAD-BLOCK CLUSTER per sample (k_cycle): the sample's angles live
 * in the cluster's distributed shared memory for the whole launch, every warp owns a fixed set of rows, and all colour
 * classes of all sweeps of all requested cycles, the fused measurement and the swap round run in ONE launch, the classes
 * separated by the hardware cluster barrier -- right when a class is a few rows per warp and a launch is latency-bound.
 * It needs R = 2 * 2^k <= 64, or_per_sweep >= 1, fused measurement, at most 12 colours, degrees <= 255 and samples small
 * enough for the shared memory of a cluster of <= 16 CTAs (else XY_ESTATE from xy_set_path / xy_run).  0 (default) =
 * automatic: path 2 where it applies, all samples' clusters are resident at once and a warp owns at most 36 rows, else
 * path 1.  Both paths give bit-identical angles, labels, accumulators and counters.  xy_get_path reports what
 * xy_run(or_per_sweep) would use (1 or 2) and the cluster size (CTAs per sample; 0 for path 1); either output may be NULL. */
int xy_set_path(xy_pt *pt, int path);
int xy_get_path(xy_pt *pt, int or_per_sweep, int *path, int *cluster_size);

/* The schedule in force: samples per launch group, and the bytes one group keeps live (its angles + its share of the
 * graph tables) -- a group that fits the 126 MB L2 is served from L2 after the first sweep of a cycle.  Either output
 * may be NULL. */
int xy_get_schedule(xy_pt *pt, int *samples_per_group, int64_t *group_bytes);

/* Tuning switches of the float2 kernel flavours (R = 2 * 2^k <= 64, R % 64 == 0); results are bit-identical for
 * every setting (tests/test_gpu_parity.py).  balance != 0: cost-balanced shares of a colour class per warp (default),
 * 0: equal shares.  pdl != 0: programmatic-dependent-launch edges between the colour-class launches (default).
 * l2_persist != 0: theta of the running sample group is marked persisting in L2 through an access-policy window
 * (default).  fuse_measure != 0: in xy_run the last over-relaxation sweep of a measured sweep also produces E, Mx, My
 * (the local field already holds cos/sin of every neighbour), 0: a separate measure launch (default on).
 * cta_shape: 0 = 32-warp CTAs (one per SM) for large colour classes and 8-warp CTAs (four per SM) for small ones
 * (default), 1 = always 8-warp, 2 = always 32-warp.  Synchronises the stream and drops the captured graphs. */
int xy_set_tuning(xy_pt *pt, int balance, int pdl, int l2_persist, int fuse_measure, int cta_shape);

/* Order of a sweep.  0 (default): the order stated at the top -- a Metropolis sweep over all
 * colours, then the over-relaxation sweep(s).  1 = INTERLEAVED: for every colour class in turn, Metropolis and then
 * over-relaxation of each of its sites (a different, equally valid Markov chain: each update leaves the Gibbs measure
 * invariant in any order).  Same-colour sites share no bond, so both updates of a site see the same neighbours and the
 * kernel serves them from ONE gather of the local field.  Needs or_per_sweep == 1 and a float2 kernel flavour
 * (R = 2 * 2^k <= 64 or R % 64 == 0), else XY_ESTATE / XY_EINVAL.  Applies to xy_run and xy_run_sweeps; xy_sweep and
 * xy_overrelax keep their meaning.  Synchronises the stream. */
int xy_set_order(xy_pt *pt, int order);

/* ---- single-colour steps (lockstep parity tests) ----
 * Metropolis on colour class `colour` of every sample with Philox sweep index `sweep` (the handle's
 * sweep counter is not touched); OR on one colour class.  Launched sample group by sample group with the
 * same grids as xy_run (xy_set_schedule), so a lockstep check exercises the timed launch configuration. */
int xy_metropolis_colour(xy_pt *pt, int colour, uint32_t sweep);
int xy_overrelax_colour(xy_pt *pt, int colour);
/* interleaved order: Metropolis (Philox sweep index `sweep`) and then over-relaxation of every site of the class */
int xy_metor_colour(xy_pt *pt, int colour, uint32_t sweep);

/* ---- state access (all synchronise the stream) ---- */
int xy_get_theta(xy_pt *pt, float *theta_host /*[S][N][R]*/);
int xy_set_theta(xy_pt *pt, const float *theta_host /*[S][N][R]*/);
/* Asynchronous upload of the whole state from PINNED host memory (cudaHostAlloc / torch pin_memory), one copy per sample
 * group of the current schedule on a second stream owned by the handle; returns at once.  theta_host must stay valid
 * and unchanged until the handle's stream has been synchronised.  The next xy_run orders each sample group's first
 * launch after that group's copy only (samples never interact, Eq. 12), so the upload of group g+1 overlaps
 * the sweeps of group g; every other call waits for the whole upload first.  Results are those of xy_set_theta. */
int xy_set_theta_async(xy_pt *pt, const float *theta_host /*[S][N][R], pinned*/);
int xy_get_labels(xy_pt *pt, int32_t *temp_of_slot_host /*[S][R]*/);
int xy_set_labels(xy_pt *pt, const int32_t *temp_of_slot_host /*[S][R], a permutation per sample*/);
/* energies per memory slot [S][R] (recomputed if stale; accumulators untouched) */
int xy_get_energy(xy_pt *pt, double *E_slot_host);
/* one swap round with the caller's decisions: accept[S][R], entry [s][t] is used for pair (t,t+1) of the
 * round's parity.  Bit-exact permutation test; round += 1. */
int xy_swap_with_decisions(xy_pt *pt, const uint8_t *accept_host);
/* accumulators [S][R][XY_NACC] indexed by temperature */
int xy_read_accumulators(xy_pt *pt, double *acc_host);
int xy_reset_accumulators(xy_pt *pt);
/* sweep / round counters and per-pair swap statistics [S][R] (entry t = pair (t,t+1)); NULLs allowed */
int xy_get_counters(xy_pt *pt, uint32_t *sweep, uint32_t *round, int64_t *swap_attempts_host,
                    int64_t *swap_accepts_host);
int xy_set_counters(xy_pt *pt, uint32_t sweep, uint32_t round);
/* device pointer of theta (caller's or the library's) */
int xy_theta_device(xy_pt *pt, float **theta_dev);
/* number of kernel launches (graph kernel nodes included) issued by this handle so far */
int xy_launch_count(xy_pt *pt, int64_t *n_launches);
int xy_synchronize(xy_pt *pt);

/* ---- diagnostic: L2 bandwidth of this GPU (the roofline denominator when a sample group is L2-resident; BASELINE.json
 * north_star "or L2 GB/s when the state fits in the 126 MB L2") ----
 * Allocates a zero-filled buffer of `bytes` (1 MiB .. 4 GiB; 32 MiB is the survey's choice, well inside L2), and times
 * `repeats` launches (CUDA events on `stream`, after two warm-up launches) of a hand-written read kernel that goes
 * through the buffer 16 times with L1 bypassed: mode 0 = linear stream of 16-byte loads, mode 1 = random aligned
 * 256-byte rows, 8 bytes per lane (the request shape of the neighbour gather at R = 64).  *gbs_out = the best launch's
 * bytes read / time in GB/s.  Runs on the current device; synchronises `stream`; frees everything it allocated. */
int xy_l2_bandwidth(size_t bytes, int mode, int repeats, void *stream /*cudaStream_t or NULL*/, double *gbs_out /*host*/);

#ifdef __cplusplus
}
#endif
#endif
