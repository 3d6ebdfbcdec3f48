// mcdc_step.cuh -- one particle segment: distances and event choice (A.2, A.4), surface event (A.5),
// collision event (A.6).  Shared by the asynchronous history kernel and the census-stepped kernel.
#pragma once
#include "mcdc_device.cuh"

namespace mcdc {

enum { LED_PRODUCTION = 0, LED_CAPTURE, LED_FISSION_ABS, LED_LEAK, LED_CENSUS_FINAL, LED_LOST, LED_N };
enum { CNT_COLL = 0, CNT_SURF, CNT_CENSUS, CNT_CHILDREN, CNT_LOST, CNT_N };

// particle state held in registers
struct PState {
  double x, y, z, ux, uy, uz, t, w;
  unsigned long long key;
  uint32_t ctr, hid;
  int g, cell, last_surf;
};

// A.2: sample d_coll, scan the cell's surfaces, compare with the distance to the census time.
// Returns the event; d = distance to it; i_star = half-space slot of the nearest surface.
__device__ __forceinline__ int find_event(const Tables &T, PState &p, double t_census, double &d, int &i_star) {
  const double INF = CUDART_INF;
  const int mat = __ldg(T.cell_mat + p.cell);
  const int mg = mat * T.G + p.g;
  const double xi = draw(p.key, p.ctr);                   // always consumed (D3)
  const double sig_t = __ldg(T.sig_t + mg);
  const double d_coll = (sig_t > 0.0) ? -log(xi) * __ldg(T.inv_sig_t + mg) : INF;
  const double ix = 1.0 / p.ux, iy = 1.0 / p.uy, iz = 1.0 / p.uz;
  double d_surf = INF;
  i_star = -1;
  const int e = __ldg(T.cell_off + p.cell + 1);
  for (int i = __ldg(T.cell_off + p.cell); i < e; ++i) {
    const int h = __ldg(T.hs + i);
    const int s = h >> 4;
    const double u = surf_distance(T, s, (h >> 1) & 7, s == p.last_surf, p.x, p.y, p.z, p.ux, p.uy, p.uz, ix, iy, iz);
    if (u < d_surf) { d_surf = u; i_star = i; }
  }
  const double d_time = __ldg(T.speed + p.g) * (t_census - p.t);
  if (d_time <= d_surf && d_time <= d_coll) { d = d_time; return EV_CENSUS; }
  if (d_surf <= d_coll) { d = d_surf; return EV_SURFACE; }
  d = d_coll;
  return EV_COLLISION;
}

// A.5 after the move.  Returns false when the particle left the problem (leak / lost).
__device__ __forceinline__ bool surface_event(const Tables &T, PState &p, int i_star, double *led_leak, double *led_lost,
                                              uint32_t *cnt_lost) {
  const int h = __ldg(T.hs + i_star);
  const int s_star = h >> 4;
  p.last_surf = s_star;
  const int bc = __ldg(T.surf_bc + s_star);
  if (bc == 1) { *led_leak += p.w; return false; }
  if (bc == 2) { reflect(T, s_star, (h >> 1) & 7, p.x, p.y, p.z, p.ux, p.uy, p.uz); return true; }
  const int c = locate_neighbour(T, i_star, s_star, p.x, p.y, p.z, p.ux, p.uy, p.uz);
  if (c < 0) { *led_lost += p.w; *cnt_lost += 1u; return false; }
  p.cell = c;
  return true;
}

// A.6.  Returns the number of fission children (>= 0) when the parent was absorbed by fission, -1 when it
// scattered (alive), -2 when it was captured.  c0 = parent's counter after the nu draw.
__device__ __forceinline__ int collision_event(const Tables &T, PState &p, uint32_t &c0, double *led_capture,
                                               double *led_fis, double *led_prod) {
  p.last_surf = -1;
  const int mat = __ldg(T.cell_mat + p.cell);
  const int mg = mat * T.G + p.g;
  const double yv = draw(p.key, p.ctr) * __ldg(T.sig_t + mg);
  const double s_tot = __ldg(T.sig_s_tot + mg);
  if (yv < s_tot) {
    const double xi_g = draw(p.key, p.ctr);
    p.g = sample_cdf(T.cdf_s + (size_t)mg * T.G, T.G, __ldg(T.last_s + mg), xi_g * s_tot);
    double xi_mu, xi_phi;
    draw2(p.key, p.ctr, xi_mu, xi_phi);
    isotropic(xi_mu, xi_phi, p.ux, p.uy, p.uz);
    return -1;
  }
  if (yv < __ldg(T.sig_sc + mg) || __ldg(T.sig_f + mg) == 0.0) { *led_capture += p.w; return -2; }
  const double xi_nu = draw(p.key, p.ctr);
  const int n = (int)floor(__ldg(T.nu + mg) + xi_nu);
  c0 = p.ctr;
  *led_fis += p.w;
  *led_prod += (double)n * p.w;
  return n;
}

// A.6 init_child: the child's own stream gives its group (chi of the fission-site material) and direction
__device__ __forceinline__ void init_child(const Tables &T, PState &p) {
  p.ctr = 0u;
  const double xi_g = draw(p.key, p.ctr);
  const int mat = __ldg(T.cell_mat + p.cell);
  p.g = sample_cdf(T.cdf_chi + (size_t)mat * T.G, T.G, __ldg(T.last_chi + mat), xi_g);
  double xi_mu, xi_phi;
  draw2(p.key, p.ctr, xi_mu, xi_phi);
  isotropic(xi_mu, xi_phi, p.ux, p.uy, p.uz);
  p.last_surf = -1;
}

// A.3 source particle of global history h.  Returns false when no cell contains it (lost).
__device__ __forceinline__ bool source_particle(const Tables &T, unsigned long long seed_mixed, unsigned long long h,
                                                PState &p) {
  p.key = mix64(seed_mixed ^ h);
  p.ctr = 0u;
  double xi_x, xi_y, xi_z, xi_t;
  draw2(p.key, p.ctr, xi_x, xi_y);
  draw2(p.key, p.ctr, xi_z, xi_t);
  const double xi_g = draw(p.key, p.ctr);
  p.x = T.src_lo[0] + xi_x * (T.src_hi[0] - T.src_lo[0]);
  p.y = T.src_lo[1] + xi_y * (T.src_hi[1] - T.src_lo[1]);
  p.z = T.src_lo[2] + xi_z * (T.src_hi[2] - T.src_lo[2]);
  p.t = T.src_t0 + xi_t * (T.src_t1 - T.src_t0);
  p.g = sample_cdf(T.src_cdf, T.G, T.src_last, xi_g);
  if (T.src_dir_mode == 0) {
    double xi_mu, xi_phi;
    draw2(p.key, p.ctr, xi_mu, xi_phi);
    isotropic(xi_mu, xi_phi, p.ux, p.uy, p.uz);
  } else {
    p.ux = T.src_dir[0]; p.uy = T.src_dir[1]; p.uz = T.src_dir[2];
  }
  p.w = 1.0;
  p.last_surf = -1;
  p.cell = locate_source(T, p.x, p.y, p.z, p.ux, p.uy, p.uz);
  return p.cell >= 0;
}

}  // namespace mcdc
