// mcdc_types.h -- plain structs shared by the host side and the kernels of libmcdc.so.
// (Product code: nothing here is shared with oracle/.)
#pragma once
#include <cstdint>

namespace mcdc {

// Surface classes recognised at mcdc_problem_create ("implementations may classify
// into typed surfaces; results must equal the general formula up to rounding").
enum SurfType : int {
  ST_PLANE_X = 0,  // q.x = position, q.y = sign of the linear coefficient
  ST_PLANE_Y = 1,
  ST_PLANE_Z = 2,
  ST_CYL_Z = 3,    // q.x = x0, q.y = y0, q.z = r^2, q.w = sign of A
  ST_QUADRIC = 4   // general 10-coefficient form (planes with a general normal included)
};

enum Event : int { EV_CENSUS = 0, EV_SURFACE = 1, EV_COLLISION = 2 };

// Particle bank in HBM, structure of arrays; index = slot * cap + i.
// Full record 92 B: x y z ux uy uz t w (8 x f64), key (u64), meta {cell, last_surface, ctr, g} (4 x i32), hid (u32).
// A fission birth record (A.6) uses x y z t w key meta.x(cell) hid = 56 B; ux/uy/uz are not allocated.
struct Bank {
  double *x, *y, *z, *ux, *uy, *uz, *t, *w;
  unsigned long long *key;
  int4 *meta;
  uint32_t *hid;
  uint32_t *count;   // [n_slots] particles stored per slot
  uint32_t *cursor;  // [n_slots] consumption cursor (transport kernel refill)
};

// Device-resident problem tables.  Every array lives in ONE contiguous blob (16-byte aligned pieces); the
// struct holds byte offsets into it, so that a kernel can address the same tables either in global memory
// (blob) or in its shared-memory copy of the blob's hot prefix (first hot_bytes bytes).
struct Tables {
  int G, M, S, C, K, Nt;
  const unsigned char *blob;   // global copy of the blob
  uint32_t hot_bytes;          // prefix a kernel may stage in shared memory (everything the hot loop reads)
  // cross sections, index mg = m * G + g
  uint32_t o_sig_t, o_inv_sig_t, o_sig_s_tot, o_sig_sc /* Sigma_s_tot + Sigma_c */, o_sig_f, o_nu;
  uint32_t o_cdf_s;     // [M*G][G] running sums of Sigma_s[m][g][.] in increasing g'
  uint32_t o_last_s;    // [M*G] last g' with a non-zero entry (fallback of the CDF scan)
  uint32_t o_cdf_chi;   // [M][G] running sums of chi
  uint32_t o_last_chi;  // [M]
  uint32_t o_speed, o_inv_speed;   // [G]
  uint32_t o_T;         // [Nt+1]
  uint32_t o_census;    // [K]
  uint32_t o_src_cdf;   // [G]
  uint32_t o_cap_frac;  // [M*G] Sigma_c / Sigma_t
  // geometry
  uint32_t o_surf_q;    // [S] double4 typed parameters
  uint32_t o_surf_bc;   // [S]
  uint32_t o_cell_off;  // [C+1]
  uint32_t o_hs;        // packed half-space: surface << 6 | bc << 4 | type << 1 | (sense > 0)
  uint32_t o_cell_mat;  // [C]
  uint32_t o_nb_off;    // [nhs+1] neighbour candidates of half-space slot i (cells across that surface)
  uint32_t o_nb_cell;
  uint32_t o_loc_off;   // [nvox+1] source locator grid
  uint32_t o_loc_cell;
  uint32_t o_cell2;     // [C] compact cell records, CELL2_BYTES each (layout below)
  uint32_t o_other2;    // "other" half-space entries, OTHER2_BYTES each
  uint32_t o_tbin_k;    // [K] int: the one time bin that holds census interval k, -1 if it spans several
  uint32_t o_it0_k;     // [K] int: time bin at the start of census interval k (hint of the general scorer)
  uint32_t o_surf_coef; // [S][10] general form (inside the hot prefix only when a general quadric exists)
  uint32_t o_rgn_off;   // [C+1] general CSG regions (Appendix J): postfix tokens of cell c, empty range = intersection
  uint32_t o_rgn_tok;   // tokens: t >= 0 half-space t of the cell's list holds; -1 AND, -2 OR, -3 NOT
  int has_regions;
  const Tables *self_dev;  // device-memory copy of this struct (slow paths that must not take the parameter's address)
  int score_fast;       // the tally mesh covers the geometry and the time grid covers [t0, C_K]: no clipping needed
  int all_one_bin;      // every cell lies in one spatial tally bin and every census interval in one time bin
  int warp_ok;          // the problem fits the compact tables of k_warp (16-bit surface / cell ids, ...)
  // techniques (include/mcdc.h mcdc_technique, DESIGN.md Appendix G); all zero = analog
  int implicit_capture;
  double wr_threshold, wr_survive;
  // source
  double src_lo[3], src_hi[3], src_t0, src_t1;
  int src_last;
  int src_dir_mode;
  int src_cell;         // >= 0: the cell of every source particle, proved at create (else -1: locate per particle):
                        //   a point source strictly inside one cell (src_chk = 0), or a source box inside the closure of
                        //   one axis-aligned box cell (src_chk = 1: valid for particles strictly inside src_clo..src_chi)
  int src_chk;
  double src_clo[3], src_chi[3];
  double src_dir[3];
  int loc_n[3];
  double loc_lo[3], loc_inv_d[3];
  // tally mesh
  double mesh_lo[3], mesh_hi[3], mesh_d[3], mesh_inv_d[3];
  int mesh_n[3];
  unsigned long long n_bins;
};

// Compact hot tables of the warp-pool kernel k_warp (built at mcdc_problem_create, staged in shared memory).
//
// Cell record, CELL2_BYTES = 40, ten 32-bit words.  The tightest axis-aligned plane of each (axis, side) is a "face"
// f = 2*axis + side (side 0 = lower bound); every other half-space of the cell (cylinders, general quadrics,
// redundant planes) is an "other".
//   +0  u16 face_surf[6]  surface id of the face (plane position = surf_q[s].x), NONE16 if the cell is unbounded there
//   +12 u16 face_nb[6]    certified neighbour cell across the face (see mcdc_host.cu "certificates"), NONE16 = search
//   +24 u8  face_idx[6]   position of the face's half-space in the cell's list (tie-break D5, generic look-ups)
//   +30 u16 face_bc       2 bits per face: boundary condition of the face's surface
//   +32 u8 n_other, u8 material, u16 other_off (first entry of the cell in the other table)
//   +36 u32 cell_bin      spatial tally bin that contains the whole cell, NONE32 if it spans several bins
// Other entry, OTHER2_BYTES = 8:
//   +0  u16 surface, u16 nb (certified neighbour across it or NONE16)
//   +4  u8 idx (position in the cell's half-space list), u8 flags = sense>0 | type<<1 | bc<<4, u16 pad
constexpr uint32_t CELL2_BYTES = 40, OTHER2_BYTES = 8;
constexpr uint32_t C2_FACE_SURF = 0, C2_FACE_NB = 12, C2_FACE_IDX = 24, C2_FACE_BC = 30, C2_INFO = 32, C2_BIN = 36;
constexpr uint32_t NONE16 = 0xFFFFu, NONE32 = 0xFFFFFFFFu;

// Per-launch parameters of the transport kernel.
struct StepParams {
  int k;                    // census index of this step (0-based); C[k] is the step's end time
  int is_last;              // k == K-1
  double t_census;          // C[k]
  int it_lo, it_n;          // time bins covered by the shared-memory tally slab
  int slab_bins;            // it_n * G * nz*ny*nx, or 0 when tallies go straight to global memory
  int n_slots;
  uint32_t cap;             // bank capacity per slot
  uint32_t hb;              // histories per slot (slot = hid / hb)
  int in_is_birth;          // input bank holds fission birth records
  int record_events;
};

// Device-side accumulators (one instance per handle).
struct DevCounters {
  double ledger[9];         // source production capture fission_abs leak census_final lost vr_gain vr_loss
  unsigned long long n[9];  // histories segments collisions surf_hits census_events children lost_n pc_removed pc_added
  int overflow;             // a bank overflowed
  int pad;
};

}  // namespace mcdc
