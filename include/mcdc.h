/* mcdc.h -- C ABI of the B200-native MC/DC hot path (libmcdc.so).
 *
 * The library runs, on one sm_100a GPU, the time-dependent multigroup Monte Carlo particle-history
 * transport loop of arXiv 2409.04668: "a fixed source problem will loop over all the particles and
 * transport them until the particle's history is terminated from a physical event (capture, fission,
 * time or space boundary), a simulation event (time census) ..." (section 2), with the
 * kernel set of PAPER.md:77 (move particle, tally, daughter particles from fission), full 3-D CSG and
 * multigroup data and hash-based, schedule-independent random numbers.
 * A problem is what the paper's input handler collects: materials and multigroup
 * cross sections, CSG surfaces and cells, a source, a tally mesh and time bins.  The quantitative
 * definition (draw order, tie-breaks, track-length estimator, batch statistics) is SURVEY.md
 * Appendix A/B as fixed in DESIGN.md.
 *
 * Conventions
 *  - Every pointer in mcdc_problem_desc and every result buffer is HOST memory owned by the caller.
 *    mcdc_problem_create deep-copies the description; the caller may free it on return.
 *  - The only DEVICE pointer crossing the boundary is the workspace handed to mcdc_workspace_bind
 *    (e.g. the data_ptr of a torch uint8 CUDA tensor) together with a CUDA stream handle
 *    (cudaStream_t as void*; NULL = default stream).  The library never frees the workspace; it
 *    must outlive every run made with it.
 *  - All real quantities are IEEE fp64; indices are int32; counters uint64.
 *  - Every call returns MCDC_OK (0) or a negative MCDC_ERR_* code; nothing throws across the ABI.
 *    A handle is not thread-safe; distinct handles are independent.
 *  - There is no CPU fallback: without a CUDA device the compute calls return MCDC_ERR_CUDA.
 */
#ifndef MCDC_H
#define MCDC_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct mcdc_problem mcdc_problem; /* opaque */

enum {
  MCDC_OK = 0,
  MCDC_ERR_ARG = -1,           /* null pointer, non-positive size, B does not divide N ...          */
  MCDC_ERR_XS = -2,            /* cross sections inconsistent (Sigma_t != Sigma_c+Sigma_s+Sigma_f,
                                  negative entries, chi not normalised where Sigma_f > 0)           */
  MCDC_ERR_GEOM = -3,          /* surface / cell / material ids out of range, empty cell            */
  MCDC_ERR_SIZE = -4,          /* result buffer size does not match the problem                     */
  MCDC_ERR_NO_WORKSPACE = -5,  /* run without a bound workspace, or workspace too small             */
  MCDC_ERR_BANK_OVERFLOW = -6, /* a particle bank overflowed; results of that run are invalid       */
  MCDC_ERR_CUDA = -7,          /* CUDA runtime error (mcdc_last_cuda_error gives the text)          */
  MCDC_ERR_NOMEM = -8,
  MCDC_ERR_GRID = -9           /* mesh / time edges / census not increasing or empty                */
};

enum { MCDC_BC_TRANSMISSION = 0, MCDC_BC_VACUUM = 1, MCDC_BC_REFLECTIVE = 2 };
enum { MCDC_DIR_ISOTROPIC = 0, MCDC_DIR_FIXED = 1 };
/* Schedulers: ASYNC = one persistent history kernel per sub-batch, census events do the
 * population bookkeeping and the particle carries on; CENSUS_STEPPED = one kernel per census step,
 * particles reaching the census time are parked in the census bank until every particle has arrived
 * (the structure a population-control step needs).                                                 */
enum { MCDC_SCHED_ASYNC = 0, MCDC_SCHED_CENSUS_STEPPED = 1 };

/* Problem description.  Layouts are C row-major.
 *  sigma_s[m][g][g2] is the transfer cross section FROM group g TO group g2.
 *  A surface is the quadric f = A x^2+B y^2+C z^2+D xy+E xz+F yz+G x+H y+I z+J (surf_coef[s][0..9]).
 *  A cell is the intersection of its half-spaces (hs_surface, hs_sense=+1 for f>0 / -1 for f<0),
 *  listed in CSR form by cell_offset[n_cells+1].  Cells must not overlap.
 *  The source is an axis-aligned box (lo==hi allowed per axis), a time interval and a group pdf.
 *  The tally mesh has mesh_n[a] uniform bins on [mesh_lo[a], mesh_hi[a]] (+-INFINITY allowed when
 *  mesh_n[a]==1), explicit time edges and all groups; bin index (((it*G+g)*nz+iz)*ny+iy)*nx+ix.
 *  census_times[n_census] is increasing; the last entry is the final time (particles stop there). */
typedef struct {
  int32_t n_groups, n_materials, n_surfaces, n_cells;
  const double *sigma_t, *sigma_c, *sigma_f, *nu, *chi; /* [M][G]                                  */
  const double *sigma_s;                                /* [M][G][G]                               */
  const double *speed;                                  /* [G] cm/s                                */
  const double *surf_coef;                              /* [S][10]                                 */
  const int32_t *surf_bc;                               /* [S] MCDC_BC_*                           */
  const int32_t *cell_offset;                           /* [C+1]                                   */
  const int32_t *hs_surface, *hs_sense;                 /* [cell_offset[C]]                        */
  const int32_t *cell_material;                         /* [C]                                     */
  double src_lo[3], src_hi[3], src_t0, src_t1;
  const double *src_group_pdf;                          /* [G]                                     */
  int32_t src_dir_mode;                                 /* MCDC_DIR_*                              */
  double src_dir[3];                                    /* unit vector when MCDC_DIR_FIXED         */
  double mesh_lo[3], mesh_hi[3];
  int32_t mesh_n[3];                                    /* nx, ny, nz                              */
  int32_t n_time_bins;
  const double *time_edges;                             /* [n_time_bins+1]                         */
  int32_t n_census;
  const double *census_times;                           /* [n_census]                              */
} mcdc_problem_desc;

/* Options of one run.  Histories first_history_id .. first_history_id+N-1 are simulated in
 * n_batches equal batches (n_batches must divide N); batch statistics per SURVEY.md A.9.        */
typedef struct {
  uint32_t n_batches;             /* >= 1                                                          */
  uint64_t first_history_id;      /* global id of the first history (resumable / shardable runs)   */
  int32_t record_history_events;  /* keep per-history event counts of this run (N x 4 uint32)      */
  int32_t scheduler;              /* MCDC_SCHED_*; both give the same trajectories and tallies      */
  /* Test knobs of the history kernel (MCDC_SCHED_ASYNC); 0 = the library chooses.  They change which
   * code path a run takes, never its results (tests/test_gpu_paths.py holds both to the oracle):
   *  debug_pool_slots: cap on the particle slots of each warp's shared-memory pool (rounded down to
   *    a multiple of 8, at least 32).  With 32 slots a pool is full after one refill and refills leave no
   *    slot free, so fission children overflow into the global ring queue in HBM by the thousand
   *    (mcdc_kernel_info_get counts them); with the default pools a handful per million do.
   *  debug_stage_tables: +1 stage the hot problem tables in shared memory whenever a pool of >= 32
   *    slots still fits; -1 never stage them (every table read goes through L1/L2).                  */
  uint32_t debug_pool_slots;
  int32_t debug_stage_tables;
} mcdc_run_opts;

typedef struct {
  /* weight ledger (A.9): source + production == capture + fission_abs + leak + census_final + lost */
  double source, production, capture, fission_abs, leak, census_final, lost;
  uint64_t histories, segments, collisions, surf_hits, census_events, children, lost_n, batches;
  uint64_t kernel_launches;       /* launches of this library's kernels since create/reset          */
  double ms_run;                  /* device time of the last mcdc_run (CUDA events on its stream)   */
  double ms_transport;            /* of which: transport kernels of the last run                    */
  /* variance reduction (mcdc_technique): weight created / removed by the weight roulette and by the
   * population control, particles the control removed / added.  The ledger then reads
   * source + production + vr_gain == capture + fission_abs + leak + census_final + lost + vr_loss
   * (to rounding: weights are no longer integers).                                                 */
  double vr_gain, vr_loss;
  uint64_t pc_removed, pc_added;
} mcdc_counters;

/* Techniques the paper names without defining them: "a variance reduction event" among the events
 * that end a flight and "time-dependent population control"; SURVEY.md
 * 8(f) NEXT-1; definition in DESIGN.md Appendix G.
 *  implicit_capture: at a collision capture += w Sigma_c/Sigma_t, w -= that, and the reaction is
 *    sampled from scatter | fission alone (y = xi (Sigma_s_tot + Sigma_f)).
 *  wr_threshold > 0: a particle that scattered with w < wr_threshold draws xi; if xi wr_survive < w it
 *    continues with w = wr_survive (wr_survive >= wr_threshold), else it dies.
 *  population_control: at every census but the last, per statistical batch, splitting-roulette to the
 *    weight w_t = W / pc_target (W = the batch's arriving weight summed in 2^-40 fixed point;
 *    pc_target = 0 means the batch's number of source histories): a particle becomes
 *    floor(w / w_t + xi) particles of weight w_t.  Needs the census-stepped scheduler (chosen
 *    automatically) and batches that fit one slot of the workspace, else MCDC_ERR_ARG.             */
typedef struct {
  int32_t implicit_capture;
  double wr_threshold, wr_survive;
  int32_t population_control;
  uint64_t pc_target;
} mcdc_technique;
/* t == NULL restores analog transport (the default).  Takes effect from the next run.              */
int mcdc_technique_set(mcdc_problem *p, const mcdc_technique *t);

/* Validates and deep-copies *d, classifies surfaces, builds cell-neighbour tables and uploads the
 * problem to the current CUDA device.  *out is untouched on error.                                */
int mcdc_problem_create(const mcdc_problem_desc *d, mcdc_problem **out);
/* General CSG regions ("full three-dimensional constructive solid geometry"; SURVEY.md 8(f)
 * NEXT-4; DESIGN.md Appendix J).  As mcdc_problem_create, but cell c is the postfix expression
 * region_rpn[region_offset[c] .. region_offset[c+1]) over its half-spaces: a token t >= 0 stands for
 * "half-space t of the cell's list holds" (0-based within the cell), MCDC_RGN_AND / _OR / _NOT combine
 * them; an empty range leaves the cell the intersection of its half-spaces.  The cell's half-space list
 * must still name every surface that bounds the cell (distances are taken to all of them).  Both
 * arrays are HOST memory, deep-copied; region_offset has n_cells + 1 entries starting at 0; expressions
 * deeper than 32 operands or malformed give MCDC_ERR_GEOM.  Both schedulers run such problems; on the
 * history kernel a region cell has no typed faces and no certified neighbours (every crossing of one
 * of its surfaces takes the cell search of A.5 with the expression evaluator).                       */
enum { MCDC_RGN_AND = -1, MCDC_RGN_OR = -2, MCDC_RGN_NOT = -3 };
int mcdc_problem_create_csg(const mcdc_problem_desc *d, const int32_t *region_offset,
                            const int32_t *region_rpn, mcdc_problem **out);
/* Universes and lattices ("full three-dimensional constructive solid geometry" is all the paper says;
 * SURVEY.md 8(f) NEXT-4; definition in DESIGN.md Appendix K).  A lattice is an nx x ny array of box elements of size
 * pitch_x x pitch_y with corner (x0, y0), all spanning z_lo .. z_hi; element (i, j) is filled with universe
 * fill[j * nx + i].  Universe u owns the quadric surfaces usurf_coef[usurf_offset[u] .. usurf_offset[u+1])[10],
 * given in coordinates LOCAL to an element (origin at the element's centre in x and y; z is not shifted), and the
 * cells ucell_offset[u] .. ucell_offset[u+1); universe cell c is the intersection of the half-spaces
 * uhs_offset[c] .. uhs_offset[c+1): uhs_surface >= 0 names a surface of the same universe (0-based within it), a
 * negative value one of the element's faces (MCDC_LAT_*), uhs_sense is +1 / -1 as in mcdc_problem_desc.
 * The flat geometry, in this order: surfaces = planes x = x0 + i pitch_x (i = 0..nx), planes y = y0 + j pitch_y
 * (j = 0..ny), z = z_lo, z = z_hi -- outer ones with bc[MCDC_LAT face order: x-lo x-hi y-lo y-hi z-lo z-hi], inner ones
 * transmission -- then element by element (j outer, i inner) the universe's surfaces translated to the element's
 * centre (f(r - c), all transmission); cells = element by element in the same order, the universe's cells in their
 * order, half-space lists in their order.  All arrays are HOST memory, deep-copied.
 *  mcdc_lattice_expand_size / mcdc_lattice_expand: the flat arrays themselves (no device needed), into caller
 *    buffers of surf_coef[S][10], surf_bc[S], cell_offset[C+1], hs_surface[H], hs_sense[H], cell_material[C].
 *  mcdc_problem_create_lattice: mcdc_problem_create on *d with its geometry fields (n_surfaces, n_cells, surf_*,
 *    cell_offset, hs_*, cell_material: ignored, may be 0 / NULL) replaced by the expansion.
 * A malformed description (universe id or local surface out of range, unknown face code, empty cell, sense not
 * +-1, non-positive pitch, z_hi <= z_lo, bc out of range) gives MCDC_ERR_GEOM.
 * Limits.  One level only: the array is two-dimensional (x, y; every element spans z_lo .. z_hi), rectangular, and a
 * universe's cells hold materials -- a cell cannot be filled with another universe or lattice (no nesting), and
 * there are no hexagonal lattices.  The expansion is a host-side flattening that copies a universe's surfaces and
 * cells into every element it fills, so the flat problem has S = nx + ny + 4 + sum over elements of the universe's
 * surfaces and C = sum over elements of its cells: memory and set-up time grow with nx * ny * |universe|.  All three
 * calls do this arithmetic in 64 bits and refuse with MCDC_ERR_GEOM a lattice whose element count nx * ny, S, C or
 * half-space count exceeds INT32_MAX.  Far below that, the history kernel's compact 16-bit tables hold fewer than
 * 65 535 cells and 65 533 surfaces: a larger flat problem still runs and still gives the same results, but on the
 * slower census-stepped kernel (mcdc_problem_info.warp_kernel_ok == 0 tells) -- a 17 x 17 lattice of pins is 578 cells,
 * a 200 x 200 one (80 000 cells) crosses the line.                                                         */
enum { MCDC_LAT_XLO = -1, MCDC_LAT_XHI = -2, MCDC_LAT_YLO = -3, MCDC_LAT_YHI = -4, MCDC_LAT_ZLO = -5, MCDC_LAT_ZHI = -6 };
typedef struct {
  int32_t n_universes;
  const int32_t *usurf_offset;             /* [U+1]                                                  */
  const double *usurf_coef;                /* [usurf_offset[U]][10], local coordinates               */
  const int32_t *ucell_offset;             /* [U+1]                                                  */
  const int32_t *uhs_offset;               /* [ucell_offset[U] + 1]                                  */
  const int32_t *uhs_surface, *uhs_sense;  /* [uhs_offset[ucell_offset[U]]]                          */
  const int32_t *ucell_material;           /* [ucell_offset[U]]                                      */
  int32_t nx, ny;
  double x0, y0, pitch_x, pitch_y, z_lo, z_hi;
  const int32_t *fill;                     /* [ny][nx] universe of element (i, j)                    */
  int32_t bc[6];                           /* MCDC_BC_* of the outer faces                           */
} mcdc_lattice_desc;
int mcdc_lattice_expand_size(const mcdc_lattice_desc *lat, int32_t *n_surfaces, int32_t *n_cells, int32_t *n_halfspaces);
int mcdc_lattice_expand(const mcdc_lattice_desc *lat, double *surf_coef, int32_t *surf_bc, int32_t *cell_offset,
                        int32_t *hs_surface, int32_t *hs_sense, int32_t *cell_material);
int mcdc_problem_create_lattice(const mcdc_problem_desc *d, const mcdc_lattice_desc *lat, mcdc_problem **out);
void mcdc_problem_destroy(mcdc_problem *p);
/* Zero tallies, ledger, census populations and counters (keeps problem and workspace).            */
int mcdc_problem_reset(mcdc_problem *p);

/* Bytes of device workspace needed to run sub-batches of up to max_histories_per_subbatch source
 * histories with up to max_batches_in_flight statistical batches resident at once (particle,
 * census and fission banks, per-batch tally accumulators).                                        */
int mcdc_workspace_size(const mcdc_problem *p, uint64_t max_histories_per_subbatch,
                        uint32_t max_batches_in_flight, size_t *bytes);
/* The smaller workspace that is enough for MCDC_SCHED_ASYNC alone (no particle banks: per-batch
 * tally accumulators and the fission queue).  A handle bound with it refuses
 * MCDC_SCHED_CENSUS_STEPPED with MCDC_ERR_NO_WORKSPACE.                                           */
int mcdc_workspace_size_async(const mcdc_problem *p, uint64_t max_histories_per_subbatch,
                              uint32_t max_batches_in_flight, size_t *bytes);
/* dev_ptr: device memory of at least `bytes` (256-byte aligned); cuda_stream: cudaStream_t.       */
int mcdc_workspace_bind(mcdc_problem *p, void *dev_ptr, size_t bytes, uint64_t max_histories_per_subbatch,
                        uint32_t max_batches_in_flight, void *cuda_stream);

/* Simulate N source histories with the 64-bit seed; accumulates into the handle's tallies and
 * ledger.  Synchronous: results are complete on return.  mcdc_run == mcdc_run_ex with one batch.  */
int mcdc_run(mcdc_problem *p, uint64_t n_histories, uint64_t seed);
int mcdc_run_ex(mcdc_problem *p, uint64_t n_histories, uint64_t seed, const mcdc_run_opts *opts);

/* k-eigenvalue mode ("k-eigenvalue and fully time-dependent simulation modes"; SURVEY.md 8(f)
 * NEXT-2; definition in DESIGN.md Appendix H): power iteration over n_inactive + n_active fission
 * generations of nominally n_particles particles.  Generation 0 is the problem's source; a generation's
 * fission children are banked, not transported; k_gen[g] = weight of the children made in generation g /
 * weight that started it; the bank is then brought to n_particles particles of weight 1 by the control
 * of mcdc_technique (splitting-roulette, each birth record drawing from its own stream).  Every active
 * generation is one statistical batch of n_particles histories of the tallies; inactive ones are
 * discarded.  Time plays no part: describe the problem with one time bin and one census far beyond any
 * flight (n_census must be 1, else MCDC_ERR_ARG: a census arrival inside a generation has no meaning here).
 * k_gen: HOST array of n_inactive + n_active doubles.  Needs the workspace of
 * mcdc_workspace_size(n_particles, 1 or more); implicit capture and roulette apply if set;
 * population_control must be off (MCDC_ERR_ARG).                                                       */
int mcdc_run_eigenvalue(mcdc_problem *p, uint64_t n_particles, uint64_t seed, uint32_t n_inactive,
                        uint32_t n_active, double *k_gen);

/* mean[i] = sum_i / N (cm of track per source history, not divided by bin volume);
 * sdev[i] = batch standard error of the mean (0 with a single batch).  n_bins must equal
 * n_time_bins*G*nz*ny*nx.                                                                          */
int mcdc_tallies_get(const mcdc_problem *p, double *mean, double *sdev, size_t n_bins);
/* mcdc_tallies_get for callers that must not allocate device memory.
 *
 * Who needs it.  mcdc_tallies_get turns the raw accumulators into mean / sdev on the GPU when the mesh is
 * large, and needs 2 * n_bins doubles of device scratch for that: it borrows them from the bound workspace
 * when that has two batch slots, and otherwise calls cudaMalloc / cudaFree.  Some hosts of this library cannot
 * live with that second case: a process that has handed all of the GPU's memory to a pooling allocator
 * (PyTorch's caching allocator, a per-rank budget fixed at job start), where a cudaMalloc made behind the pool's
 * back fails or eats into what the pool was promised; and a read-out inside a timing-critical loop, where
 * cudaMalloc and cudaFree make the host wait for everything else the device is doing.
 *
 * What it does.  The same A.9 statistics by the same kernel (identical results to mcdc_tallies_get), with the
 * scratch in a fixed array that lives inside libmcdc.so's device image: 2 * MCDC_NOALLOC_MAX_BINS doubles = 16 MiB.
 * Every GPU on which the process uses the library holds those 16 MiB from the moment the library's device
 * code is loaded there until the process exits, whether or not this call is ever made.  The call itself
 * makes no cudaMalloc, cudaFree or other allocating CUDA / library call: one kernel launch, two device-to-host
 * copies on the bound stream (or the default stream if none is bound), one stream synchronisation.  A bound
 * workspace is not needed and not touched.
 *
 *  mean, sdev: HOST arrays of n_bins doubles owned by the caller (pinned or pageable), layout and meaning of
 *    mcdc_tallies_get; complete on return.
 *  n_bins: must equal the problem's bin count (else MCDC_ERR_SIZE) and must not exceed MCDC_NOALLOC_MAX_BINS:
 *    a larger mesh is refused with MCDC_ERR_SIZE and mcdc_last_cuda_error() then says so in words -- nothing
 *    is launched, and nothing is silently truncated.  (Config 2's 7.2e6-bin mesh is beyond it; bind a
 *    workspace with two slots and use mcdc_tallies_get there.)
 *  MCDC_ERR_ARG before the first run (no histories), or if the GPU that holds the handle is not the
 *    calling thread's current device.
 *
 * First call on each GPU: the library looks up the array's device address (cudaGetSymbolAddress, with that
 * GPU current) and remembers it for the life of the process.  That look-up may make the runtime load the
 * library's device code onto the GPU, so make the first call per GPU at start-up, before any stream capture
 * begins anywhere in the process; later calls only launch, copy and wait.
 *
 * Sharing.  There is ONE array per GPU per process, shared by every handle, stream and thread.  It keeps
 * whatever the previous call left in it; that is harmless here because each call overwrites the first n_bins
 * entries of both halves before it copies them out, so nothing has to be cleared between calls.  But two calls
 * whose GPU work can overlap (two host threads reading out two handles on different streams of the same
 * GPU) write the same memory and corrupt each other's results: serialise them yourself.  Calls made one
 * after another from one thread never overlap, since each waits for its stream before returning.        */
#define MCDC_NOALLOC_MAX_BINS ((size_t)1 << 20)
int mcdc_tallies_get_noalloc(const mcdc_problem *p, double *mean, double *sdev, size_t n_bins);
/* Collision-estimator tally, the paper's one code listing (Fig. 3:
 * `add(mcdc.col_tally, part.v, loc2index(part))` inside tally_collision_event); SURVEY.md 8(f) NEXT-4;
 * reading in DESIGN.md Appendix I: at every collision the bin of the SAME mesh that holds the collision
 * site (r, t, g) takes w / Sigma_t, w the weight the particle arrives with -- an estimate of the same flux
 * as the track-length tally.  Off by default; enable before the run.  The accumulators are allocated by
 * the library (one per batch slot of the bound workspace); while the tally is enabled its sum / sumsq are part
 * of the mcdc_state_export vector (every rank must then have it enabled).
 * mcdc_collision_tallies_get has the layout and statistics of mcdc_tallies_get.                        */
int mcdc_collision_tally_enable(mcdc_problem *p, int on);
int mcdc_collision_tallies_get(const mcdc_problem *p, double *mean, double *sdev, size_t n_bins);
/* Raw accumulators: sum over batches of S_b and of S_b^2.                                          */
int mcdc_tally_sums_get(const mcdc_problem *p, double *sum, double *sumsq, size_t n_bins);
int mcdc_counters_get(const mcdc_problem *p, mcdc_counters *c);
/* Population bookkeeping at census: summed weight and number of particles that reached census k.  */
int mcdc_census_get(const mcdc_problem *p, double *pop_w, uint64_t *pop_n, size_t n_census);
/* Weight and number of particles that LEFT the population control at census k (zero where none ran). */
int mcdc_census_after_get(const mcdc_problem *p, double *pop_w, uint64_t *pop_n, size_t n_census);
/* ev[h][0..3] = collisions, surface events, fission children, census events of history
 * first_history_id+h of the LAST run (needs record_history_events).                               */
int mcdc_history_events_get(const mcdc_problem *p, uint32_t *ev, size_t n_histories);

/* What mcdc_problem_create derived from the geometry: how many transmission
 * half-spaces have a certified neighbour, how many cells lie in one spatial tally bin, the bytes of
 * tables the history kernel stages in shared memory, and whether the problem fits that kernel's
 * compact tables at all (else MCDC_SCHED_CENSUS_STEPPED is used).                                 */
typedef struct {
  uint64_t transmission_halfspaces, certified_halfspaces, cells, one_bin_cells, hot_table_bytes;
  int32_t warp_kernel_ok, score_fast;
  int32_t all_one_bin;   /* every cell in one spatial tally bin and every census interval in one time bin: the
                            history kernel without the 4-D DDA scorer is used                               */
  int32_t source_cell;   /* >= 0: the cell source particles are born in without a search -- a point source
                            proved strictly inside it, or a source box inside the closure of this axis-aligned
                            box cell (particles drawn strictly inside its bounds); -1: search per particle    */
} mcdc_problem_info;
int mcdc_problem_info_get(const mcdc_problem *p, mcdc_problem_info *info);

/* Multi-GPU domain replication (PAPER.md:59 "domain-replicated MPI", :173-177):
 * every rank runs its own history-id range on a full copy of the problem, and the raw accumulators are
 * summed over ranks once at the end.  These calls expose the handle's accumulators as ONE fp64 vector
 * so that the caller can reduce it with any collective (ncclAllReduce on a device buffer, gloo/MPI on
 * a host buffer) and put the sum back:
 *   [0, n_bins) sum   [n_bins, 2 n_bins) sumsq   [then sum and sumsq of the collision-estimator tally, 2 n_bins
 *   more entries, while mcdc_collision_tally_enable is on]   then, in exactly this order, pop_w[K], pop_n[K],
 *   ledger[9] (source production capture fission_abs leak census_final lost vr_gain vr_loss),
 *   counts[9] (histories segments collisions surf_hits census_events children lost_n pc_removed pc_added),
 *   histories, batches -- so with T = (2 or 4) n_bins + 2 K: vr_gain is entry T + 7, segments T + 10, pc_added
 *   T + 17, histories (the handle's total, what mean / sdev divide by) T + 18, batches T + 19.
 * Integer entries are stored as doubles (exact below 2^53).  on_device != 0: buf is DEVICE memory
 * (copies run on the bound stream, synchronous on return); else HOST memory.  n must equal
 * mcdc_state_size.  Import REPLACES the handle's accumulators; ranks must use the same batch size. */
int mcdc_state_size(const mcdc_problem *p, size_t *n_doubles);
int mcdc_state_export(const mcdc_problem *p, double *buf, size_t n_doubles, int on_device);
int mcdc_state_import(mcdc_problem *p, const double *buf, size_t n_doubles, int on_device);

/* Which transport kernel the LAST run of this handle launched, as text: the k_warp instantiation
 * "k_warp<STAGED,RECORD,VARIANT,SCORE,threads>", the revision of the kernel sources it was built from (first
 * 12 hex digits of their SHA-1, set by the build), the grid, the pool slots per warp and the dynamic shared
 * memory, and the number of fission children that have gone through the global ring queue since the handle was
 * created ("queue_children=N": evidence that a run took the overflow path) -- or "k_transport ..." for the
 * census-stepped scheduler; empty before the first run.  Measurement
 * aid: bench.py keys the ncu-derived constants of profiles/ by this string, so a figure
 * captured from another kernel build is never printed beside this one's timing.  buf: HOST, n bytes,
 * always NUL-terminated; MCDC_ERR_ARG on NULL / n == 0.                                              */
int mcdc_kernel_info_get(const mcdc_problem *p, char *buf, size_t n);

const char *mcdc_strerror(int code);
const char *mcdc_last_cuda_error(const mcdc_problem *p);
/* "major.minor sm_XX" of the build; never fails.                                                  */
const char *mcdc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MCDC_H */
