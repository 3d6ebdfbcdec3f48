// mcdc_step.cuh -- one particle segment: flight initialisation (A.3 / A.6 sampling of group and direction),
// distances and event choice (A.2, A.4), surface event (A.5), collision event (A.6).
// Shared by the asynchronous history kernel and the census-stepped kernel.
#pragma once
#include "mcdc_device.cuh"

namespace mcdc {

enum { LED_PRODUCTION = 0, LED_CAPTURE, LED_FISSION_ABS, LED_LEAK, LED_CENSUS_FINAL, LED_LOST, LED_VR_GAIN, LED_VR_LOSS, LED_N };
enum { CNT_COLL = 0, CNT_SURF, CNT_CENSUS, CNT_CHILDREN, CNT_LOST, CNT_N };

// what a lane still has to sample before its particle can fly (draw order of A.3 / A.6 is kept per particle)
enum FlightInit : int {
  FI_NONE = 0,
  FI_SCATTER = 1,   // outgoing group from the scatter row of (material, incoming group), then isotropic direction
  FI_CHILD = 2,     // group from chi of the fission-site material, then isotropic direction
  FI_SOURCE = 3     // group from the source pdf, direction (isotropic or fixed), then cell location
};

// particle state held in registers
struct PState {
  double x, y, z, ux, uy, uz, t, w;
  double ix, iy, iz;                // 1 / (ux, uy, uz), kept with the direction (history kernel only)
  unsigned long long key;
  uint32_t ctr, hid;
  int g, cell, last_surf;
};

// first index with xi < cdf[i]; fallback `last`.  cdf(i) is any callable.
template <class F>
__device__ __forceinline__ int sample_cdf(F cdf, int n, int last, double xi) {
#pragma unroll 1
  for (int i = 0; i < n; ++i)
    if (xi < cdf(i)) return i;
  return last;
}

// Common tail of source birth (A.3), child birth (A.6 init_child) and scattering (A.6): one draw for the
// group, two for the direction.  All lanes that need it run it together.  Returns false when a source
// particle is in no cell (lost).
template <class TBT>
__device__ __forceinline__ bool flight_init(const TBT &tb, PState &p, int kind) {
  const Tables &T = tb.T;
  const double xi_g = draw(p.key, p.ctr);
  if (kind == FI_SCATTER) {
    const int mg = tb.cell_mat(p.cell) * T.G + p.g;
    const int row = mg * T.G;
    p.g = sample_cdf([&](int i) { return tb.cdf_s(row + i); }, T.G, tb.last_s(mg), xi_g * tb.sig_s_tot(mg));
  } else if (kind == FI_CHILD) {
    const int mat = tb.cell_mat(p.cell);
    const int row = mat * T.G;
    p.g = sample_cdf([&](int i) { return tb.cdf_chi(row + i); }, T.G, tb.last_chi(mat), xi_g);
  } else {
    p.g = sample_cdf([&](int i) { return tb.src_cdf(i); }, T.G, T.src_last, xi_g);
  }
  if (kind == FI_SOURCE && T.src_dir_mode != 0) {
    p.ux = T.src_dir[0]; p.uy = T.src_dir[1]; p.uz = T.src_dir[2];
  } else {
    double xi_mu, xi_phi;
    draw2(p.key, p.ctr, xi_mu, xi_phi);
    isotropic(xi_mu, xi_phi, p.ux, p.uy, p.uz);
  }
  p.ix = 1.0 / p.ux; p.iy = 1.0 / p.uy; p.iz = 1.0 / p.uz;
  p.last_surf = -1;
  if (kind == FI_SOURCE) {
    p.cell = locate_source<true>(tb, p.x, p.y, p.z, p.ux, p.uy, p.uz);
    return p.cell >= 0;
  }
  return true;
}

// A.3, first part: key, position and time of the source particle of global history h (draws xi_x..xi_t);
// group, direction and cell follow in flight_init(FI_SOURCE).
__device__ __forceinline__ void source_position(const Tables &T, unsigned long long seed_mixed, unsigned long long h,
                                                PState &p) {
  p.key = mix64(seed_mixed ^ h);
  p.ctr = 0u;
  double xi_x, xi_y, xi_z, xi_t;
  draw2(p.key, p.ctr, xi_x, xi_y);
  draw2(p.key, p.ctr, xi_z, xi_t);
  p.x = T.src_lo[0] + xi_x * (T.src_hi[0] - T.src_lo[0]);
  p.y = T.src_lo[1] + xi_y * (T.src_hi[1] - T.src_lo[1]);
  p.z = T.src_lo[2] + xi_z * (T.src_hi[2] - T.src_lo[2]);
  p.t = T.src_t0 + xi_t * (T.src_t1 - T.src_t0);
  p.w = 1.0;
  p.last_surf = -1;
  p.cell = -1;
}

// smallest k with C[k] > t, else K-1 (D15)
template <class TBT>
__device__ __forceinline__ int census_index(const TBT &tb, double t) {
#pragma unroll 1
  for (int k = 0; k < tb.T.K; ++k)
    if (tb.census(k) > t) return k;
  return tb.T.K - 1;
}

// A.2: sample d_coll, scan the cell's surfaces, compare with the distance to the census time.
// Returns the event; d = distance to it; i_star = half-space slot of the nearest surface.
template <class TBT>
__device__ __forceinline__ int find_event(const TBT &tb, PState &p, double t_census, double &d, int &i_star) {
  const double INF = CUDART_INF;
  const int mg = tb.cell_mat(p.cell) * tb.T.G + p.g;
  const double xi = draw(p.key, p.ctr);                   // always consumed (D3)
  const double sig_t = tb.sig_t(mg);
  const double d_coll = (sig_t > 0.0) ? -log(xi) * tb.inv_sig_t(mg) : INF;
  const double ix = 1.0 / p.ux, iy = 1.0 / p.uy, iz = 1.0 / p.uz;
  double d_surf = INF;
  i_star = -1;
  const int e = tb.cell_off(p.cell + 1);
  for (int i = tb.cell_off(p.cell); i < e; ++i) {
    const int h = tb.hs(i);
    const int s = h >> 6;
    const double u = surf_distance(tb, s, (h >> 1) & 7, s == p.last_surf, p.x, p.y, p.z, p.ux, p.uy, p.uz, ix, iy, iz);
    if (u < d_surf) { d_surf = u; i_star = i; }
  }
  const double d_time = tb.speed(p.g) * (t_census - p.t);
  if (d_time <= d_surf && d_time <= d_coll) { d = d_time; return EV_CENSUS; }
  if (d_surf <= d_coll) { d = d_surf; return EV_SURFACE; }
  d = d_coll;
  return EV_COLLISION;
}

// A.5 after the move.  Returns false when the particle left the problem (leak / lost).
template <class TBT>
__device__ __forceinline__ bool surface_event(const TBT &tb, PState &p, int i_star, double *led_leak, double *led_lost,
                                              uint32_t *cnt_lost) {
  const int h = tb.hs(i_star);
  const int s_star = h >> 6;
  p.last_surf = s_star;
  const int bc = tb.surf_bc(s_star);
  if (bc == 1) { *led_leak += p.w; return false; }
  if (bc == 2) { reflect(tb, s_star, (h >> 1) & 7, p.x, p.y, p.z, p.ux, p.uy, p.uz); return true; }
  const int c = locate_neighbour<true>(tb, i_star, s_star, p.x, p.y, p.z, p.ux, p.uy, p.uz);
  if (c < 0) { *led_lost += p.w; *cnt_lost += 1u; return false; }
  p.cell = c;
  return true;
}

// A.6 reaction choice, with the techniques of Appendix G when the problem asks for them.  Returns -1: scattered
// (the caller must run flight_init(FI_SCATTER) before the next segment); -2: dead (captured, or killed by the
// weight roulette); n >= 0: absorbed by fission with n children, c0 = parent's counter after the nu draw.
template <class TBT>
__device__ __forceinline__ int collision_event(const TBT &tb, PState &p, uint32_t &c0, double *led_capture,
                                               double *led_fis, double *led_prod, double *led_gain, double *led_loss) {
  const Tables &T = tb.T;
  p.last_surf = -1;
  const int mg = tb.cell_mat(p.cell) * T.G + p.g;
  const double xi = draw(p.key, p.ctr);
  const double s_tot = tb.sig_s_tot(mg), sig_f = tb.sig_f(mg);
  bool scatter;
  if (T.implicit_capture) {                                // G.1
    const double w_c = p.w * tb.cap_frac(mg);
    *led_capture += w_c;
    p.w -= w_c;
    const double s_r = s_tot + sig_f;
    if (!(s_r > 0.0)) { *led_capture += p.w; p.w = 0.0; return -2; }
    scatter = (xi * s_r < s_tot) || sig_f == 0.0;
  } else {
    const double yv = xi * tb.sig_t(mg);
    scatter = yv < s_tot;
    if (!scatter && (yv < tb.sig_sc(mg) || sig_f == 0.0)) { *led_capture += p.w; return -2; }
  }
  if (scatter) {
    if (T.wr_threshold > 0.0 && p.w < T.wr_threshold) {    // G.2
      const double xi_r = draw(p.key, p.ctr);
      if (xi_r * T.wr_survive < p.w) { *led_gain += T.wr_survive - p.w; p.w = T.wr_survive; }
      else { *led_loss += p.w; return -2; }
    }
    return -1;
  }
  const double xi_nu = draw(p.key, p.ctr);
  const int n = (int)floor(tb.nu(mg) + xi_nu);
  c0 = p.ctr;
  *led_fis += p.w;
  *led_prod += (double)n * p.w;
  return n;
}

}  // namespace mcdc
