// mcdc_typed.cuh -- the hot-loop versions of A.2/A.4 (distances), A.5 (surface event) and A.7 (track-length
// scoring) on the typed cell records built at mcdc_problem_create (mcdc_types.h, CELL_REC_BYTES).
//
// A cell is {axis-aligned faces} + {other half-spaces}.  For a face axis the forward plane is picked by the sign
// of the direction component: the backward plane of the axis has a negative distance (rejected by A.4's "> 0"
// rule) and the plane just crossed is always a backward one, so this equals A.4's scan over both planes for any
// particle inside its cell.  The other half-spaces use the generic routines.
#pragma once
#include "mcdc_step.cuh"

namespace mcdc {

// A.2 on a typed cell.  Returns the event; d = distance to it; slot_star = half-space slot of the nearest surface
// (valid when the event is EV_SURFACE); pos_star = plane position when that surface is a face (else unused);
// which = 2*axis + side for a face, 6 for an "other" surface.
template <class TBT>
__device__ __forceinline__ int find_event_typed(const TBT &tb, PState &p, double t_census, double &d, int &slot_star,
                                                int &which, double &pos_star) {
  const double INF = CUDART_INF;
  const uint32_t rec = tb.T.o_cell_rec + (uint32_t)p.cell * CELL_REC_BYTES;
  const int mg = tb.template ldb<int>(rec + CR_MAT) * tb.T.G + p.g;
  const double xi = draw(p.key, p.ctr);                   // always consumed (D3)
  const double sig_t = tb.sig_t(mg);
  const double d_coll = (sig_t > 0.0) ? -log(xi) * tb.inv_sig_t(mg) : INF;

  // ---- faces: one candidate per axis ----
  const int fx = (p.ux > 0.0) ? 1 : 0, fy = (p.uy > 0.0) ? 3 : 2, fz = (p.uz > 0.0) ? 5 : 4;
  const double px = tb.template ldb<double>(rec + CR_BOUND + 8u * fx);
  const double py = tb.template ldb<double>(rec + CR_BOUND + 8u * fy);
  const double pz = tb.template ldb<double>(rec + CR_BOUND + 8u * fz);
  const double dx = (px - p.x) * p.ix, dy = (py - p.y) * p.iy, dz = (pz - p.z) * p.iz;   // 0 * inf = NaN: rejected
  double d_surf = INF;
  which = -1;
  pos_star = 0.0;
  if (dx > 0.0 && dx < INF) { d_surf = dx; which = fx; pos_star = px; }
  if (dy > 0.0 && dy <= d_surf && dy < INF) {
    // equal distances (an edge hit): the earlier half-space of the cell's list wins (D5)
    if (dy < d_surf || tb.template ldb<int>(rec + CR_FACE + 4u * fy) < tb.template ldb<int>(rec + CR_FACE + 4u * which)) {
      d_surf = dy; which = fy; pos_star = py;
    }
  }
  if (dz > 0.0 && dz <= d_surf && dz < INF) {
    if (dz < d_surf || tb.template ldb<int>(rec + CR_FACE + 4u * fz) < tb.template ldb<int>(rec + CR_FACE + 4u * which)) {
      d_surf = dz; which = fz; pos_star = pz;
    }
  }
  // ---- other half-spaces (cylinders, general quadrics, redundant planes), list order, strict < ----
  slot_star = -1;
  const int n_other = tb.template ldb<int>(rec + CR_N_OTHER);
  if (n_other > 0) {
    const int2 o01 = tb.template ldb<int2>(rec + CR_OTHER0);
    const int ooff = tb.template ldb<int>(rec + CR_OTHER_OFF);
    for (int j = 0; j < n_other; ++j) {
      const int slot = (j == 0) ? o01.x : ((j == 1) ? o01.y : tb.template ldb<int>(tb.T.o_other + 4u * (uint32_t)(ooff + j)));
      const int h = tb.hs(slot);
      const int s = h >> 6;
      const double u = surf_distance(tb, s, (h >> 1) & 7, s == p.last_surf, p.x, p.y, p.z, p.ux, p.uy, p.uz, p.ix, p.iy, p.iz);
      if (u < d_surf) { d_surf = u; which = 6; slot_star = slot; }
    }
  }
  const double d_time = tb.speed(p.g) * (t_census - p.t);
  if (d_time <= d_surf && d_time <= d_coll) { d = d_time; return EV_CENSUS; }
  if (d_surf <= d_coll) {
    d = d_surf;
    if (which < 6) slot_star = tb.template ldb<int>(rec + CR_FACE + 4u * which);
    return EV_SURFACE;
  }
  d = d_coll;
  return EV_COLLISION;
}

// a coordinate exactly on face f of the typed cell at `rec`: the direction rule of A.3 decides (generic routine, rare)
template <class TBT>
__device__ __forceinline__ bool face_tie(const TBT &tb, uint32_t rec, int f, int s_star, const PState &p) {
  const int slot = tb.template ldb<int>(rec + CR_FACE + 4u * (uint32_t)f);
  if (slot < 0) return false;                              // NaN coordinate against an infinite bound
  const int h = tb.hs(slot);
  const int s = h >> 6, want = (h & 1) ? 1 : -1;
  return surf_sense(tb, s, (h >> 1) & 7, s == s_star, p.x, p.y, p.z, p.ux, p.uy, p.uz) == want;
}

// Does typed cell c contain r for a particle moving along u that has just crossed surface s_star (A.5)?
// crossed_axis >= 0: s_star is an axis-aligned plane at pos_star on that axis.  The particle's coordinate on that
// axis equals pos_star only up to rounding, so that bound is decided by the direction (D11): the cell lists
// (s_star, opposite sense), hence its tightest bound behind the particle is pos_star -- or lies beyond it, and
// then the cell does not touch the crossed plane.
template <class TBT>
__device__ __forceinline__ bool cell_contains_typed(const TBT &tb, int c, int s_star, int crossed_axis, double pos_star,
                                                    const PState &p) {
  const uint32_t rec = tb.T.o_cell_rec + (uint32_t)c * CELL_REC_BYTES;
  const double r[3] = {p.x, p.y, p.z}, o[3] = {p.ux, p.uy, p.uz};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double lo = tb.template ldb<double>(rec + CR_BOUND + 16u * a);
    const double hi = tb.template ldb<double>(rec + CR_BOUND + 16u * a + 8u);
    bool chk_lo = true, chk_hi = true;
    if (a == crossed_axis) {
      if (o[a] > 0.0) { if (lo != pos_star) return false; chk_lo = false; }
      else            { if (hi != pos_star) return false; chk_hi = false; }
    }
    if (chk_lo && !(r[a] > lo)) {
      if (r[a] < lo) return false;
      if (!face_tie(tb, rec, 2 * a, s_star, p)) return false;
    }
    if (chk_hi && !(r[a] < hi)) {
      if (r[a] > hi) return false;
      if (!face_tie(tb, rec, 2 * a + 1, s_star, p)) return false;
    }
  }
  const int n_other = tb.template ldb<int>(rec + CR_N_OTHER);
  if (n_other > 0) {
    const int2 o01 = tb.template ldb<int2>(rec + CR_OTHER0);
    const int ooff = tb.template ldb<int>(rec + CR_OTHER_OFF);
    for (int j = 0; j < n_other; ++j) {
      const int slot = (j == 0) ? o01.x : ((j == 1) ? o01.y : tb.template ldb<int>(tb.T.o_other + 4u * (uint32_t)(ooff + j)));
      const int h = tb.hs(slot);
      const int s = h >> 6, want = (h & 1) ? 1 : -1;
      if (surf_sense(tb, s, (h >> 1) & 7, s == s_star, p.x, p.y, p.z, p.ux, p.uy, p.uz) != want) return false;
    }
  }
  return true;
}

// A.5 after the move, typed.  Returns false when the particle left the problem (leak / lost).
template <class TBT>
__device__ __forceinline__ bool surface_event_typed(const TBT &tb, PState &p, int slot_star, int which, double pos_star,
                                                    double *led_leak, double *led_lost, uint32_t *cnt_lost) {
  const int h = tb.hs(slot_star);
  const int s_star = h >> 6, bc = (h >> 4) & 3, type = (h >> 1) & 7;
  p.last_surf = s_star;
  if (bc == 1) { *led_leak += p.w; return false; }
  if (bc == 2) {
    if (type == ST_PLANE_X) { p.ux = -p.ux; p.ix = -p.ix; }
    else if (type == ST_PLANE_Y) { p.uy = -p.uy; p.iy = -p.iy; }
    else if (type == ST_PLANE_Z) { p.uz = -p.uz; p.iz = -p.iz; }
    else {
      reflect(tb, s_star, type, p.x, p.y, p.z, p.ux, p.uy, p.uz);
      p.ix = 1.0 / p.ux; p.iy = 1.0 / p.uy; p.iz = 1.0 / p.uz;
    }
    return true;
  }
  const int crossed_axis = (which < 6) ? (which >> 1) : -1;
  int c = -1;
  const int e = tb.nb_off(slot_star + 1);
  for (int i = tb.nb_off(slot_star); i < e; ++i) {
    const int cand = tb.nb_cell(i);
    if (cell_contains_typed(tb, cand, s_star, crossed_axis, pos_star, p)) { c = cand; break; }
  }
  if (c < 0) c = locate_all(tb, s_star, p.x, p.y, p.z, p.ux, p.uy, p.uz);
  if (c < 0) { *led_lost += p.w; *cnt_lost += 1u; return false; }
  p.cell = c;
  return true;
}

}  // namespace mcdc
