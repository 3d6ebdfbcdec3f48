/* mcdc_oracle.h -- C interface of the ORACLE (test infrastructure, not product).
 *
 * A plain, slow, single-threaded CPU restatement of the time-dependent multigroup Monte Carlo
 * particle-history transport loop of arXiv 2409.04668 (PAPER.md:75 fixed-source loop; PAPER.md:77
 * move / tally / fission-daughter kernels; PAPER.md:59 CSG + multigroup + time-dependent;
 * PAPER.md:61 hash-based RNG), in the reading fixed by SURVEY.md Appendix A/B/D and DESIGN.md.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * load this library.  It shares no code, header or table with the CUDA path (include/mcdc.h,
 * paper_2409_04668_b200/csrc/); the struct below is deliberately its own type.
 */
#ifndef MCDC_ORACLE_H
#define MCDC_ORACLE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_problem orc_problem;

typedef struct {
  int32_t G, M, S, C;                 /* groups, materials, surfaces, cells                  */
  const double *sigma_t, *sigma_c, *sigma_f, *nu, *chi; /* [M][G]                            */
  const double *sigma_s;              /* [M][G][G], from g to g'                             */
  const double *speed;                /* [G]                                                 */
  const double *surf_coef;            /* [S][10]  A B C D E F G H I J                        */
  const int32_t *surf_bc;             /* [S] 0 transmission, 1 vacuum, 2 reflective          */
  const int32_t *cell_offset;         /* [C+1]                                               */
  const int32_t *hs_surface, *hs_sense; /* [cell_offset[C]]                                  */
  const int32_t *cell_material;       /* [C]                                                 */
  double src_lo[3], src_hi[3], src_t0, src_t1;
  const double *src_group_pdf;        /* [G]                                                 */
  int32_t src_dir_mode;               /* 0 isotropic, 1 fixed                                */
  double src_dir[3];
  double mesh_lo[3], mesh_hi[3];
  int32_t mesh_n[3];                  /* nx ny nz                                            */
  int32_t Nt;  const double *time_edges;   /* [Nt+1]                                         */
  int32_t K;   const double *census;       /* [K]                                            */
} orc_desc;

typedef struct {
  double source, production, capture, fission_abs, leak, census_final, lost;
  uint64_t histories, segments, collisions, surf_hits, census_events, children, lost_n, batches;
  /* variance reduction (Appendix G of DESIGN.md): weight created / removed by weight roulette and by the
   * population control at census, and the particles the control removed / added                         */
  double vr_gain, vr_loss;
  uint64_t pc_removed, pc_added;
} orc_counters;

/* Techniques named by the paper ("a variance reduction event"; "time-dependent
 * population control"), in the reading of DESIGN.md Appendix G:
 *  implicit_capture: at a collision capture += w Sigma_c/Sigma_t, w -= that, and the reaction is sampled
 *    from scatter | fission alone (y = xi (Sigma_s_tot + Sigma_f));
 *  weight roulette: a particle that scattered with w < wr_threshold draws xi; xi wr_survive < w keeps it
 *    with w = wr_survive, else it dies;
 *  population_control (splitting-roulette) at every census but the last, per statistical batch: with
 *    W = sum over the batch's arrivals of trunc(w 2^40) 2^-40 and w_t = W / pc_target, a particle becomes
 *    n = floor(w / w_t + xi) particles of weight w_t (copy 0 keeps its stream, copy j >= 1 takes the
 *    stream child_key(key, ctr after xi, j)).                                                          */
typedef struct {
  int32_t implicit_capture;
  double wr_threshold, wr_survive;       /* wr_threshold <= 0: no roulette                       */
  int32_t population_control;
  uint64_t pc_target;                    /* 0: the number of source histories of the batch        */
} orc_technique;

typedef struct {
  uint32_t n_batches;         /* B, must divide n_histories                                  */
  uint64_t first_history_id;
  int32_t record_history_events;
  int32_t bank_fifo;          /* 0: LIFO secondary bank (default), 1: FIFO   (pin E5)        */
  int32_t reverse_histories;  /* 1: process each batch's histories in decreasing id (pin E5) */
} orc_run_opts;

int  orc_create(const orc_desc *d, orc_problem **out);   /* deep copy; 0 or negative error   */
/* General CSG regions ("full three-dimensional constructive solid geometry"; DESIGN.md Appendix J):
 * cell c becomes the postfix expression region_rpn[region_offset[c] .. region_offset[c+1]) over its half-spaces
 * (token t >= 0: "half-space t of the cell's list holds"; -1 AND, -2 OR, -3 NOT); an empty range leaves the cell
 * the intersection of its half-spaces.  The cell's list still names every surface that bounds it.            */
int  orc_regions_set(orc_problem *p, const int32_t *region_offset, const int32_t *region_rpn);
int  orc_technique_set(orc_problem *p, const orc_technique *t);   /* NULL: analog (the default)        */
void orc_destroy(orc_problem *p);
void orc_reset(orc_problem *p);
int  orc_run(orc_problem *p, uint64_t n_histories, uint64_t seed, const orc_run_opts *o);
/* k-eigenvalue mode (DESIGN.md Appendix H): n_inactive + n_active fission generations of nominally
 * N particles; k_gen[g] = children weight / starting weight of generation g; active generations are the
 * statistical batches of the tallies.  reverse_order: process each generation's bank backwards (pin H-d).  */
int  orc_run_eigenvalue(orc_problem *p, uint64_t N, uint64_t seed, uint32_t n_inactive, uint32_t n_active,
                        int32_t reverse_order, double *k_gen);
int  orc_tallies_get(const orc_problem *p, double *mean, double *sdev, size_t n_bins);
int  orc_tally_sums_get(const orc_problem *p, double *sum, double *sumsq, size_t n_bins);
/* collision-estimator tally of the paper's Fig. 3 (DESIGN.md Appendix I): off by default */
int  orc_collision_tally_enable(orc_problem *p, int on);
int  orc_collision_tallies_get(const orc_problem *p, double *mean, double *sdev, size_t n_bins);
int  orc_counters_get(const orc_problem *p, orc_counters *c);
int  orc_census_get(const orc_problem *p, double *pop_w, uint64_t *pop_n, size_t K);
int  orc_history_events_get(const orc_problem *p, uint32_t *ev /* [n][4] */, size_t n);
/* weight and number of particles that left the population control at census k (zero where no control ran) */
int  orc_census_after_get(const orc_problem *p, double *pop_w, uint64_t *pop_n, size_t K);

/* unit-level entry points used by the pins (tests/test_oracle_*.py) */
uint64_t orc_mix64(uint64_t z);
uint64_t orc_source_key(uint64_t seed, uint64_t h);
uint64_t orc_child_key(uint64_t parent_key, uint32_t c0, uint32_t j);
void     orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void     orc_draws(uint64_t key, uint32_t first_ctr, size_t n, double *out);
double   orc_surface_distance(const double coef[10], const double r[3], const double omega[3], int on_surface);
int      orc_locate(const orc_problem *p, const double r[3], const double omega[3]);
/* advance one particle from (r, omega, cell) through surface events only (no collisions, no time limit):
 * returns the number of surface events performed (<= max_events); writes final r, omega, cell.         */
int      orc_stream(const orc_problem *p, double r[3], double omega[3], int32_t *cell, int max_events);
/* score one straight segment into the current batch accumulator (A.7) and close the batch */
int      orc_score_segment(orc_problem *p, const double r[3], const double omega[3], double t, int g,
                           double w, double d);
int      orc_close_batch(orc_problem *p, uint64_t histories_in_batch);
/* the population control of G.3 applied to a bank given as arrays: n_out[i] = copies made of particle i */
int      orc_population_control(orc_problem *p, size_t n, const double *w, const uint64_t *key, const uint32_t *ctr,
                                uint64_t target, int32_t *n_out, double *w_t_out);

#ifdef __cplusplus
}
#endif
#endif
