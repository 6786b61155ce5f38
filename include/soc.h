/*
 * soc.h -- C ABI of libsoc_b200: the per-frequency photon-package simulation of SOC's Monte Carlo
 * radiative transfer (Juvela, arXiv:1812.06632) and the energy-balance temperature kernel, as
 * hand-written CUDA for sm_100a.
 *
 * Citations are lines of the paper text and readings S1-S17 of DESIGN.md where the paper is
 * silent.  What the calls compute:
 *   - the model is a regular Cartesian root grid of cubic cells with octree refinement; all cells form ONE
 *     vector: root cells first, then level 2, ... (Sect. 2.1.1)
 *   - one kernel simulates the photon packages of ONE frequency; it sees the densities, the optical depth
 *     of that frequency and a per-cell absorption counter; the host loops over frequencies
 *   - packages come from an isotropic external background and from blackbody point sources
 *
 *   - the absorbed energy integrated over frequency is turned into dust temperatures by a separate kernel;
 *     cells that were never hit get a constant temperature
 *
 * Conventions
 *   - every function returns SOC_OK (0) or a negative error code; the text of the last error of the calling
 *     thread is available from soc_last_error().  No exception or abort crosses the boundary.
 *   - pointers are HOST memory unless the comment says DEVICE.  Host arrays are borrowed for the duration
 *     of the call only; the library never frees or keeps caller memory.  DEVICE arrays are caller-owned.
 *   - lengths are in units of the root-cell edge ("GL").  Cell order of every per-cell array is the paper's
 *     cell vector: level 1 (root, index = ix + nx*(iy + ny*iz)), then level 2, ...; the 8 cells of an octet
 *     are consecutive with slot = bx + 2*by + 4*bz (reading S5).
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - there is no CPU fallback: without a CUDA device every compute call fails with SOC_ECUDA.
 */
#ifndef SOC_B200_H
#define SOC_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SOC_OK      0
#define SOC_EINVAL (-1)   /* bad argument or inconsistent hierarchy */
#define SOC_ENOMEM (-2)   /* host or device allocation failed */
#define SOC_ECUDA  (-3)   /* CUDA runtime error; text in soc_last_error() */

#define SOC_MAX_POINT_SOURCES 64
#define SOC_MAX_LEVELS 16

/* flags of the simulate calls */
#define SOC_GEOM_FP32 0u  /* production: fp32 package state (in-cell position, direction, remaining optical depth) evaluated
                             in fp32; fp32 package weight relative to the initial energy; deposits summed per launch in an
                             internal fp32 accumulator (fp64 with option "acc32" = 0) that is folded into the caller's fp64
                             array after every frequency */
#define SOC_GEOM_FP64 1u  /* replay: the same fp32 package state, every update evaluated in fp64 and rounded once; fp64
                             weight; fp64 atomic adds straight into the caller's array; per-package records.
                             Same decisions as the oracle's fp32-state variant except within 2^-29 of a rounding boundary */

/* opaque; owns its device copies of the cloud and the dust tables, its internal accumulators and result slots.
 * A grid serves ONE stream and ONE host thread at a time: calls on the same grid must be issued in stream order from one
 * thread (the internal accumulators, result slots and the staged temperature table are per grid, not per call).  Use one
 * grid per stream for concurrent work.  soc_grid_create returns with the grid complete (device synchronised). */
typedef struct soc_grid soc_grid;

/* Inputs named by the paper: the cloud hierarchy with the density values, the dust cross sections for
 * absorption and scattering, the scattering function per frequency (here Henyey-Greenstein g,
 * north_star).  Single dust population. */
typedef struct {
    int32_t nx, ny, nz;         /* root grid */
    int32_t n_levels;           /* n_L >= 1; 1 = regular grid; <= SOC_MAX_LEVELS */
    const int64_t *n_cells;     /* [n_levels]; n_cells[0] = nx*ny*nz, the others multiples of 8; sum < 2^31 */
    const float *density;       /* [n_total] level-major; leaves finite and >= 0; parents ignored */
    const int32_t *child;       /* [n_total]: -1 = leaf, else index WITHIN level l+1 of the first cell of the
                                   cell's octet (multiple of 8).  NULL when n_levels == 1 */
    int32_t n_freq;
    const double *freq_hz;      /* [n_freq] strictly ascending (index 0 = lowest frequency) */
    const double *kabs, *ksca;  /* [n_freq] optical depth per unit density per GL, >= 0 */
    const double *g;            /* [n_freq] Henyey-Greenstein asymmetry, |g| < 1 */
} soc_grid_desc;

/* Radiation sources at one frequency.  Package ids [0, n_bg) are background
 * packages of energy pi*I*S/n_bg (S = surface of the root grid); id p >= n_bg belongs to point source
 * (p - n_bg) mod n_point and carries L_k / count_k (reading S3). */
typedef struct {
    double bg_intensity;        /* I_nu of the isotropic background; 0 = none */
    int32_t n_point;            /* <= SOC_MAX_POINT_SOURCES */
    const double *ps_pos;       /* [n_point][3], GL, strictly inside the root grid; a source may sit in an
                                   empty cell */
    const double *ps_lum;       /* [n_point] L_nu in the same energy unit as pi*I*S */
    int64_t n_bg;               /* -1 = default split: all packages to the only class present, n/2 each if both */
    const double *beam;         /* test hook, normally NULL: [6] = position, unit direction; every package is
                                   this beam with energy 1 and no random emission */
    /* Dust re-emission (row f1; PAPER.md:67 "the emission is calculated by SOC itself", :79, :143): the LAST n_dust
     * package ids are emitted by the cells -- uniform point in the cell, isotropic direction.  Cell c sends
     * dust_count[c] packages of energy L_c / dust_count[c], L_c = 4 pi kabs rho_c h^3 B_nu(T_c) at the frequency of
     * the call; consecutive ids are spread over the cells (id -> id * stride mod n_dust).  n_bg and the default split
     * refer to the first n_packages - n_dust ids. */
    int64_t n_dust;             /* 0 = none; must equal the sum of dust_count and be < 2^32 */
    const float *dust_T;        /* DEVICE [n_total] dust temperature per cell (what soc_update_temperatures wrote) */
    const int32_t *dust_count;  /* DEVICE [n_total] packages per cell (soc_emission_counts, or the caller's own policy);
                                   0 wherever L_c = 0 */
    double *dust_self;          /* DEVICE [n_total] or NULL (row f3): += weight * the energy a cell's own packages deposit
                                   in it before they first leave it -- the absorption-emission cycle inside a cell that
                                   the diagonal ALI operator takes out of the iteration */
} soc_sources;

typedef struct {
    double emitted, escaped, absorbed;   /* energies of the simulated packages (not multiplied by `weight`) */
    uint64_t cell_steps, scatterings, terminated;
    double weight_drift;                 /* production mode: max over the escaped packages of |w - (1 - sum of deposits)|,
                                            the fp32 running weight against the deposits actually made, both relative to
                                            the package's initial energy (escaped is taken from the deposits while less than
                                            half was absorbed, so emitted = absorbed + escaped does not see this drift);
                                            replay mode: 0 (fp64 weight, deposit = weight difference) */
    uint64_t gather_requests, red_requests;   /* option "stats" = 1, production mode: global-memory gather instructions
                                            (cell words, reverse links) and reduction instructions (red.global.add) the
                                            lanes issued -- the request counts behind bench.py's roofline.components;
                                            0 otherwise */
    uint64_t suspensions, queue_refusals;     /* slab-blocked launches (option "slabs"): package states written to a queue
                                            (slab crossings and end-of-phase hand-overs), and packages a full queue
                                            refused, which walked on unconfined; 0 otherwise */
} soc_freq_result;

/* per-package replay record (DEVICE array written by soc_simulate_packages) */
typedef struct {
    uint64_t hash;              /* h = 0xcbf29ce484222325; per cell-step h = (h ^ cell id) * 0x100000001b3 */
    uint32_t steps, scatters;
    double e_escaped;           /* weight with which the package left the grid (0 if terminated) */
} soc_replay_record;

/* Copies and validates the model (child indices in range and multiples of 8, every octet has exactly one
 * parent, leaf densities finite and >= 0, dust tables finite).  On success *out owns device memory until
 * soc_grid_destroy. */
int soc_grid_create(const soc_grid_desc *desc, soc_grid **out);
void soc_grid_destroy(soc_grid *grid);
int64_t soc_grid_n_total(const soc_grid *grid);

/* Quadrature weights of the frequency integral (trapezoid in nu, reading S9): w[n_freq]. */
int soc_freq_weights(const soc_grid *grid, double *w);

/* Simulate package ids [0, n_packages) at frequency index ifreq (rows a1-a9 of the scope table):
 *   absorbed[cell] += weight * (energy absorbed in the cell)     DEVICE, n_total doubles, accumulated into
 * Philox4x32-10 stream keyed by (seed, ifreq, package id) (north_star; reading S2).  `res` (may be NULL)
 * receives the totals; when it is non-NULL the call synchronises the stream before returning, otherwise it
 * only enqueues work. */
int soc_simulate_frequency(soc_grid *grid, int32_t ifreq, const soc_sources *src, int64_t n_packages,
                           uint64_t seed, double weight, double *absorbed, soc_freq_result *res,
                           uint32_t flags, void *cuda_stream);

/* Replay / subset entry: package ids [pkg_begin, pkg_begin + pkg_count) of the same run (package energies
 * depend on the full n_packages).  `replay` (DEVICE, pkg_count records) may be NULL. */
int soc_simulate_packages(soc_grid *grid, int32_t ifreq, const soc_sources *src, int64_t n_packages,
                          uint64_t seed, double weight, int64_t pkg_begin, int64_t pkg_count,
                          double *absorbed, soc_replay_record *replay, soc_freq_result *res,
                          uint32_t flags, void *cuda_stream);

/* Frequency loop (row a10): for every frequency f of the grid, packages
 * [pkg_begin, pkg_begin + pkg_count) of n_packages with sources src[f], accumulated as
 *   absorbed_int[cell] += w_f * A_f[cell]            (w = soc_freq_weights)
 * All launches are queued back to back on the stream; results[n_freq] (may be NULL) are fetched once at
 * the end (the call then synchronises).  Sources with dust packages (n_dust > 0 at any frequency) are accepted; such a
 * spectrum is served one frequency at a time whatever option "overlap" says (the offsets of the dust packages exist once
 * per grid) and synchronises the stream once per frequency. */
int soc_simulate_spectrum(soc_grid *grid, const soc_sources *src, int64_t n_packages, uint64_t seed,
                          int64_t pkg_begin, int64_t pkg_count, double *absorbed_int,
                          soc_freq_result *results, uint32_t flags, void *cuda_stream);

/* Package counts of the dust re-emission (row f1).  mode 0 "the same number of photon packages is sent
 * per each cell", the total a multiple of the number of emitting cells: m = ceil(n_request / n_emitting) from every
 * cell with L_c > 0.  mode 1 "weighted according to the emission" with "the maximum number of photon packages sent
 * from any single cell ... limited": n_c = min(cap, ceil(n_request L_c / sum L)), at least 1 where L_c > 0.
 * T: DEVICE n_total floats.  count: DEVICE n_total int32, written.  *n_dust (HOST) receives the sum; *lum_total (HOST,
 * may be NULL) the sum of the L_c.  Synchronises the stream. */
int soc_emission_counts(soc_grid *grid, int32_t ifreq, const float *T, int32_t mode, int64_t n_request, int32_t cap,
                        int32_t *count, int64_t *n_dust, double *lum_total, void *cuda_stream);

/* Frequency-integrated emission of every cell, emitted[c] = sum_f w_f L_c,f(T_c) (w = soc_freq_weights): what the cell
 * radiates in a dust simulation at these temperatures -- the denominator of the ALI escape probability.
 * T: DEVICE n_total floats; emitted: DEVICE n_total doubles, written. */
int soc_cell_emission(soc_grid *grid, const float *T, double *emitted, void *cuda_stream);

/* Temperature update with the diagonal ALI operator (row f3; "solves explicitly for the cycle of photons
 * that are absorbed within the emitting cell ... one additional floating point number per cell ... to keep track of
 * the photon escape probabilities").  beta_c = self_abs[c] / emitted[c] (clamped to [0, 0.999]); the table is entered
 * with E = scale (absorbed[c] - self_abs[c]) / (rho h^3 (1 - beta_c)); beta = 0 is soc_update_temperatures.
 * absorbed, self_abs, emitted: DEVICE n_total doubles of the same simulation(s). */
int soc_update_temperatures_ali(soc_grid *grid, const double *absorbed, const double *self_abs, const double *emitted,
                                double scale, const float *table_T, int32_t n_table, double E_min, double E_max,
                                float *T_out, void *cuda_stream);

/* soc_update_temperatures_ali for callers that cannot allocate GPU memory at the time of the call.  Same operation, same
 * arguments, same result (row f3), but the call makes no cudaMalloc / cudaMallocHost / cudaFree and takes
 * nothing from the library's buffer cache.
 *
 * Who needs it.  soc_update_temperatures_ali allocates on its first use per grid: a per-cell work array on the device and
 * a pinned staging buffer for the table.  That is a problem for a host program that
 *   - has handed the whole device to an allocator of its own (a framework's caching pool sized to all of HBM, a service
 *     with a fixed memory budget per tenant): a cudaMalloc from inside this library then fails, or takes memory the
 *     program has not accounted for;
 *   - runs the temperature update inside a loop that must not stall: cudaMalloc and cudaFree synchronise the whole
 *     device, so a first-use allocation in iteration k stops every other stream of the process for its duration;
 *   - must prove at start-up that the run cannot die of memory exhaustion half-way through.
 *
 * How it works.  The work array and the table sit in an array that is compiled into the library
 * (static __device__, 16 MiB + 32 KiB).  Every GPU on which the library's module is loaded holds that array until the
 * process exits, used or not -- that is the price.  The limit it sets: grids of at most 2 097 152 cells in total
 * (soc_grid_n_total; a 128^3 regular grid fits exactly) and n_table <= 8192.  A larger grid is refused with SOC_EINVAL
 * and a message that names both numbers; nothing is launched in that case.
 *
 * Set-up.  The first call on each device looks up the device address of the array (cudaGetSymbolAddress) and remembers
 * it; later calls on that device only launch.  Make that first call during start-up, before any CUDA stream capture is
 * begun.  The grid's device must be the current device (SOC_EINVAL otherwise).
 *
 * Sharing.  There is ONE array per GPU, shared by every grid, stream and host thread of the process, and it keeps what
 * the last call wrote.  Nothing in it needs clearing between calls: each call overwrites the elements it later reads.
 * But two calls whose kernels can run on the GPU at the same time (different streams without an event between them,
 * different host threads) write the same elements and corrupt each other's temperatures -- order them yourself.  Calls
 * issued on one stream are ordered by the stream.
 *
 * absorbed, self_abs, emitted: DEVICE n_total doubles (no alignment requirement).  T_out: DEVICE n_total floats, 16-byte
 * aligned, written.  table_T: HOST n_table floats; pageable memory is read before the call returns, page-locked memory
 * is read when the stream reaches the copy and must stay unchanged until then.  The call only enqueues work. */
int soc_update_temperatures_ali_static(soc_grid *grid, const double *absorbed, const double *self_abs,
                                       const double *emitted, double scale, const float *table_T, int32_t n_table,
                                       double E_min, double E_max, float *T_out, void *cuda_stream);

/* Iterated run with dust re-emission (rows f1, f3):
 *   iteration 0   the constant sources src[f] (background, point sources), n_const packages per frequency, `seed`:
 *                 A_const = sum_f w_f A_f;  T = table(A_const)
 *   iteration i   1 .. n_iter: for every frequency the cells emit n_request[i-1] packages (counts by `mode`, `cap` from
 *                 the current T), seed + i:  D_i = sum_f w_f A_dust,f
 *                 reference field: R_i = mean of D_k, k = ref_start .. i, weighted by n_request[k-1]
 *                 (R_i = D_i without it and for i < ref_start);  T = table(A_const + R_i), through the ALI update if ali
 * n_request may change from iteration to iteration.  absorbed_out (DEVICE n_total doubles) receives
 * A_const + R of the last iteration, T_out (DEVICE n_total floats) the temperatures; history (HOST, may be NULL):
 * [n_iter + 1] records.  Synchronises. */
typedef struct {
    int32_t mode, cap;          /* package counts: soc_emission_counts */
    int32_t reference_field;    /* 0 / 1 */
    int32_t ref_start;          /* first iteration that enters the running mean (>= 1) */
    int32_t ali;                /* 0 / 1 */
    int32_t n_iter;
    const int64_t *n_request;   /* HOST [n_iter] */
} soc_iterate_opts;

typedef struct {
    double emitted, escaped, absorbed;   /* frequency-integrated (sum_f w_f ...) energies of the iteration's packages */
    int64_t n_packages;                  /* packages simulated in the iteration, all frequencies */
    uint64_t cell_steps;
} soc_iterate_record;

int soc_iterate(soc_grid *grid, const soc_sources *src, int64_t n_const, uint64_t seed, const soc_iterate_opts *opts,
                double t_scale, const float *table_T, int32_t n_table, double E_min, double E_max,
                double *absorbed_out, float *T_out, soc_iterate_record *history, uint32_t flags, void *cuda_stream);

/* Surface-brightness map at frequency index ifreq (row f2; PAPER.md:55 K3, :67 "a mapping kernel to make surface brightness
 * maps for the desired frequencies and directions", :137).  Thermal dust emission integrated along parallel lines of
 * sight with extinction by absorption + scattering, no background, no scattered light (reading M1):
 *     I = sum over the cells k crossed, front to back:  exp(-tau_k) kabs/(kabs+ksca) B_nu(T_k) (1 - exp(-dtau_k)),
 *     dtau_k = (kabs + ksca) rho_k ds_k.
 * Pixel (i, j), i fastest, looks along `dir` from  centre + ((i+1/2) - npx/2) pixel ex + ((j+1/2) - npy/2) pixel ey;
 * ex, ey, dir orthonormal (checked to 1e-6), lengths in root-cell edges (reading M2).  T: DEVICE n_total floats.
 * map: DEVICE npx*npy floats, written (intensity in the unit of B_nu, cgs). */
typedef struct {
    double ex[3], ey[3], dir[3], centre[3];
    int32_t npx, npy;
    double pixel;
} soc_map_desc;

int soc_make_map(soc_grid *grid, int32_t ifreq, const float *T, const soc_map_desc *desc, float *map, void *cuda_stream);

/* Energy balance by table lookup (row a11; reading S10).  For every leaf with rho > 0:
 *   E = scale * absorbed[cell] / (rho * h^3),  h = 2^-(level-1)
 *   T = table_T interpolated linearly in the index x = (ln E - ln E_min)/(ln E_max - ln E_min)*(n_table-1);
 *   E <= E_min (also cells never hit) -> table_T[0];  E >= E_max -> table_T[n_table-1].
 * Parent cells and rho = 0 leaves get 0.  table_T: HOST, n_table floats (2 <= n_table <= 8192).
 * absorbed: DEVICE n_total doubles.  T_out: DEVICE n_total floats. */
int soc_update_temperatures(soc_grid *grid, const double *absorbed, double scale, const float *table_T,
                            int32_t n_table, double E_min, double E_max, float *T_out, void *cuda_stream);

/* End-to-end entry with HOST buffers only: uploads the model, zeroes a device accumulator, runs
 * soc_simulate_spectrum for seeds seed, seed+1, ... seed+n_iter-1 (running mean over iterations, reading
 * S12), updates the temperatures, and copies absorbed_int (mean over iterations, n_total doubles) and
 * T (n_total floats) back.  Either output pointer may be NULL.  results: [n_iter][n_freq] or NULL. */
int soc_run_host(const soc_grid_desc *desc, const soc_sources *src, int64_t n_packages, uint64_t seed,
                 int32_t n_iter, double t_scale, const float *table_T, int32_t n_table, double E_min,
                 double E_max, double *absorbed_int_out, float *T_out, soc_freq_result *results,
                 uint32_t flags);

/* Tuning knobs (all have defaults chosen for B200): "blocks_per_sm", "threads", "refill_threshold" (replay
 * kernel), "service_threshold" (parked lanes that trigger a service pass), "hot_cache" (0/1: shared partial sums
 * for the cells around point sources), "stats" (0/1: the production kernels count their gather and reduction
 * instructions, and the 16-byte loads / stores of queued package states, into soc_freq_result; a slower kernel variant,
 * for measurement runs), "acc32" (0/1: fp32 per-launch accumulator), "overlap" (0/1: soc_simulate_spectrum overlaps consecutive frequencies on two streams), "kernel" (production kernel on
 * regular grids: 0 = chosen by working-set size, 1 = photon_fast_kernel, 2 = photon_q_kernel), "carveout"
 * (preferred shared-memory carve-out in %, -1 = driver default), "slabs" (regular grids whose cell words + fp32
 * accumulator exceed L2: number of z-slabs a frequency is served in -- a package that crosses a slab boundary waits in a
 * device queue for that slab's turn; 0 = by working-set size, 1 = off; the queues take 52 bytes x packages of the launch
 * x slabs of device memory per accumulator set), "slab_sweeps" (sweeps over the slabs before the last, whole-grid launch
 * of a frequency; 0 = 2), "slab_queue_limit" (test hook: entries a slab / leftover queue accepts from the walk before it
 * refuses packages; 0 = its capacity), "slab_chunk" (test hook: packages per sequence of phases, 0 = 2^24: a frequency of
 * more packages is served in several sequences), "group" (soc_simulate_spectrum: consecutive frequencies per launch where
 * a frequency has few packages -- one launch then carries the packages of up to 4 frequencies, each lane reading the
 * opacities of its package's frequency, into one internal accumulator with the quadrature weights folded into the package
 * energies; 0 = by package count (up to ~1.6e7 packages per launch) for background-only sources, 1 = off, 2-4 = that
 * many also with point sources, where the shared fp32 accumulator costs accuracy near the sources: cells against counters
 * 6e-7 instead of 3e-8 on config 3; constant sources only, grids served by photon_fast_kernel, frequencies whose package
 * energies lie within 1e-7 (1e-2 with point sources) of the brightest of the launch); and
 * "timing" (0/1): record a CUDA-event pair on the launching stream around every photon-kernel launch.
 * Returns SOC_EINVAL for an unknown key or an out-of-range value. */
int soc_set_option(soc_grid *grid, const char *key, int64_t value);

/* With option "timing" = 1: ms[i] = device time of the photon kernel last launched into result slot i
 * (slot = frequency index for soc_simulate_spectrum, 0 for the single-frequency calls); -1 where no launch
 * was recorded.  soc_simulate_spectrum overlaps consecutive launches on two streams (option "overlap", default 1)
 * and gives a launch of few packages up to four consecutive frequencies (option "group"): there the time of a launch is
 * the advance of the completion front (end of this launch - end of the one before, so that the sum is the span from the
 * first start to the last end), and the frequencies of two consecutive launches share the time of both equally.  Waits
 * for those launches to finish.  ms: HOST, n floats. */
int soc_get_timings(soc_grid *grid, int32_t n, float *ms);

/* Roofline probes: random 4-byte gathers (kind 0), random fp64 red.global.add (kind 1),
 * random fp32 red.global.add (kind 2), random 32-byte gathers (kind 3: one sector = a 2x2x2 brick of fp32 cells),
 * random 16-byte red.global.add.v4.f32 (kind 4), random 16-byte gathers (kind 6: half a brick), and the memory side of
 * one cell-step (kind 5: a 4-byte gather from the first half of the footprint and an fp32 red.global.add at the same
 * random cell of the second half) over a
 * footprint of `footprint_bytes`, n_ops operations in total, uniform addresses, no arithmetic, every access
 * independent of the others.  A footprint of a few hundred cells is the hot-spot case (many threads
 * updating "a small number of cells close to the source"): kinds 1 and 2 over 343 cells give the rate of contended
 * global reductions, and kind 7 the rate of the remedy the photon kernels use there -- fp32 atomic adds into a
 * shared-memory copy of the cells (at most 8192 cells = 32 KB footprint), one fp64 red.global.add per touched cell and
 * block at the end.  *ms receives the CUDA-event time of the probe kernel. */
int soc_probe_throughput(int32_t kind, int64_t footprint_bytes, int64_t n_ops, float *ms);

/* Stochastically heated grains (row f4; Appendix A -- a companion solver, "not part of SOC" proper).
 * Per cell and grain size the fraction p_i of grains in each enthalpy bin solves R p = 0, sum p = 1, where "the upward
 * transitions (R_ji, i < j) are obtained by taking a vector product of the intensity with the integration weights", "the
 * pre-calculated cooling rates occupy the elements R_(i-1,i)", the diagonal follows from detailed balance and all other
 * elements are zero, so that "the linear equations can be solved efficiently with forward-substitutions" (:361).  The
 * emission is emission[cell][f] = sum_s abundance[s] sum_i p[cell][s][i] emis[s][i][f].
 * The integration weights are given in the sparse form they have in practice: a photon of frequency f takes a grain of bin
 * i to ONE bin jup[s][i][f] (-1: none) at the rate wup[s][i][f] * intensity[f].
 * All model arrays: HOST, copied by soc_stochastic_create.  n_e <= 128, n_freq <= 1024. */
typedef struct soc_stochastic soc_stochastic;
typedef struct {
    int32_t n_size, n_e, n_freq;
    const int32_t *jup;         /* [n_size][n_e][n_freq]  target bin, > i, or -1 */
    const double *wup;          /* [n_size][n_e][n_freq]  weight of that transition */
    const double *cool;         /* [n_size][n_e]          cooling rate i -> i - 1 (element 0 unused), > 0 */
    const double *emis;         /* [n_size][n_e][n_freq]  emission of one grain in bin i */
    const double *abundance;    /* [n_size] */
} soc_stochastic_model;

int soc_stochastic_create(const soc_stochastic_model *model, soc_stochastic **out);
void soc_stochastic_destroy(soc_stochastic *model);

/* intensity: DEVICE [n_cells][n_freq] doubles.  emission: DEVICE [n_cells][n_freq] doubles, written.  p_out: DEVICE
 * [n_cells][n_size][n_e] doubles or NULL. */
int soc_stochastic_emission(soc_stochastic *model, const double *intensity, int64_t n_cells, double *emission,
                            double *p_out, void *cuda_stream);

/* Bounds-checked build (libsoc_b200_checked.so, compiled with -DSOC_CHECKED): number of out-of-range indices the photon
 * kernels produced so far in this process (each such access was redirected to element 0), after synchronising the device.
 * -1 in the product library, where the checks are compiled out.  -2 on a CUDA error. */
int64_t soc_checked_violations(void);

/* Number of kernel launches issued by this library in the calling process (bench.py's "gpu_launches"). */
uint64_t soc_launch_count(void);

/* The package queues of slab-blocked launches (option "slabs": ~1 GB per accumulator set for 1e7 packages in two slabs)
 * and the large per-grid device arrays (cell words, links, accumulators) outlive the grid that allocated them:
 * soc_grid_destroy hands them to a process-wide cache (two queue buffers; per-grid arrays up to 8 GB in total), from which
 * the next grid takes buffers of the same size (soc_run_host creates a grid per call; cudaMalloc / cudaFree of buffers
 * this size cost it tens to hundreds of milliseconds, differently every time).  This call frees the cache (device
 * synchronised).  Returns the number of bytes released.  The library makes the same call itself when one of its device
 * allocations fails, and then tries that allocation once more, so idle cached buffers never cause SOC_ENOMEM.  The 8 GB
 * limit of the per-grid array cache can be set in the environment: SOC_B200_CACHE_MB (megabytes, read once; 0 = cache
 * nothing). */
int64_t soc_release_cached_memory(void);

const char *soc_last_error(void);
const char *soc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SOC_B200_H */
