// mcdc_host.cu -- C ABI (include/mcdc.h) of libmcdc.so: validation, problem upload, the census-step
// driver loop and result read-back.  All transport arithmetic runs in the kernels of mcdc_kernels.cuh.
#include <algorithm>
#include <array>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/mcdc.h"
#include "mcdc_warp_inst.cuh"

using namespace mcdc;

namespace {

const double HINF = std::numeric_limits<double>::infinity();

struct DeviceArena {           // device allocations owned by the handle
  std::vector<void *> ptrs;
  cudaError_t err = cudaSuccess;
  template <class V>
  const V *upload(const std::vector<V> &h) {
    void *d = nullptr;
    size_t bytes = std::max<size_t>(h.size(), 1) * sizeof(V);
    cudaError_t e = cudaMalloc(&d, bytes);
    if (e != cudaSuccess) { err = e; return nullptr; }
    ptrs.push_back(d);
    if (!h.empty()) {
      e = cudaMemcpy(d, h.data(), h.size() * sizeof(V), cudaMemcpyHostToDevice);
      if (e != cudaSuccess) err = e;
    }
    return (const V *)d;
  }
  template <class V>
  V *zeros(size_t n) {
    void *d = nullptr;
    size_t bytes = std::max<size_t>(n, 1) * sizeof(V);
    cudaError_t e = cudaMalloc(&d, bytes);
    if (e != cudaSuccess) { err = e; return nullptr; }
    ptrs.push_back(d);
    e = cudaMemset(d, 0, bytes);
    if (e != cudaSuccess) err = e;
    return (V *)d;
  }
  void release() {
    for (void *p : ptrs) cudaFree(p);
    ptrs.clear();
  }
};

struct Box { double lo[3], hi[3]; };

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace

#ifndef MCDC_KERNEL_REV
#define MCDC_KERNEL_REV "unknown"      // build.py: first 12 hex digits of the SHA-1 over the kernel sources
#endif

struct mcdc_problem {
  // host copy of the description (deep)
  int G, M, S, C, K, Nt;
  std::vector<double> sigma_t, sigma_c, sigma_f, nu, chi, sigma_s, speed, surf_coef, src_pdf, T, census;
  std::vector<int> surf_bc, cell_off, hs_surface, hs_sense, cell_mat;
  std::vector<int> rgn_off, rgn_tok;   // general CSG regions (Appendix J): postfix expression per cell, empty = intersection
  double src_lo[3], src_hi[3], src_t0, src_t1, src_dir[3];
  int src_dir_mode;
  double mesh_lo[3], mesh_hi[3];
  int mesh_n[3];
  size_t n_bins, n_spatial;
  // device
  DeviceArena arena;
  Tables tab;
  double *d_sum = nullptr, *d_sumsq = nullptr, *d_pop_w = nullptr, *d_pop_w_after = nullptr;
  unsigned long long *d_pop_n = nullptr, *d_pop_n_after = nullptr;
  // collision-estimator tally (Appendix I): handle-owned, allocated when it is switched on
  int col_on = 0;
  double *d_xc_acc = nullptr, *d_sumc = nullptr, *d_sumsqc = nullptr;
  uint32_t xc_slots = 0;
  unsigned long long *d_wfix = nullptr;   // [ws_slots] arriving weight of a batch in 2^-40 fixed point (workspace)
  mcdc_technique tech = {0, 0.0, 0.0, 0, 0ull};
  DevCounters *d_cnt = nullptr;
  uint32_t *d_ev = nullptr;      // [n][4] of the last run (cudaMalloc'ed on demand, kept and grown)
  size_t ev_n = 0, ev_cap = 0;
  // workspace (caller-owned)
  char *ws = nullptr;
  size_t ws_bytes = 0;
  uint64_t ws_hist = 0;
  uint32_t ws_slots = 0;
  uint32_t cap = 0;              // bank capacity per slot
  cudaStream_t stream = nullptr;
  Bank bankA, bankB, bankS1, bankS2;
  double *x_acc = nullptr;
  uint32_t *counts_dev = nullptr;
  FissionQueue queue;
  uint32_t *d_hist_cursor = nullptr;   // handle-owned
  unsigned long long *d_head_tail = nullptr;
  // bookkeeping
  uint64_t histories = 0, batches = 0, batch_size = 0, launches = 0;
  double ms_run = 0.0, ms_transport = 0.0;
  int n_sm = 148, blocks_per_sm = 1, blocks_per_sm_hist = 1;
  bool stage_tables = false;
  int hist_threads = 512;
  uint32_t pool_slots = 0, pool_reserve = 0;
  size_t pool_smem = 0;
  size_t n_cert = 0, n_transm = 0, n_one_bin = 0;   // certified / all transmission half-spaces; cells in one tally bin
  // CUDA events owned by the handle (created on first use, destroyed with it): run brackets, one pair per
  // k_warp launch of the run in flight (ev_used of them recorded), the pair around each k_transport launch
  cudaEvent_t e_run0 = nullptr, e_run1 = nullptr, e_tr0 = nullptr, e_tr1 = nullptr;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev_pairs;
  size_t ev_used = 0;
  // census-step mode of k_warp: pinned snapshot of the live counts + overflow flag, looked at a few steps late (run_subbatch_stepwarp)
  uint32_t *h_poll = nullptr;
  size_t h_poll_cap = 0;
  cudaEvent_t e_poll = nullptr;
  bool transport_attr_set = false;   // cudaFuncSetAttribute(k_transport) done for this handle's device
  std::string last_kernel;           // transport kernel instantiation + launch shape of the last run (mcdc_kernel_info_get)
  std::string cuda_err;
};

namespace {

int ensure_collision_buffers(mcdc_problem *p);   // defined with the result calls
int batch_statistics(mcdc_problem *p, const double *d_sum, const double *d_sumsq, double *mean, double *sdev, size_t n_bins);

int cuda_fail(mcdc_problem *p, cudaError_t e, const char *where) {
  p->cuda_err = std::string(where) + ": " + cudaGetErrorString(e);
  return MCDC_ERR_CUDA;
}
#define CK(call)                                                     \
  do {                                                               \
    cudaError_t e__ = (call);                                        \
    if (e__ != cudaSuccess) return cuda_fail(p, e__, #call);         \
  } while (0)

// ---------------------------------------------------------------------------------------------
// validation
// ---------------------------------------------------------------------------------------------
int validate(const mcdc_problem_desc *d) {
  if (!d) return MCDC_ERR_ARG;
  if (d->n_groups < 1 || d->n_materials < 1 || d->n_surfaces < 1 || d->n_cells < 1) return MCDC_ERR_ARG;
  if (!d->sigma_t || !d->sigma_c || !d->sigma_f || !d->nu || !d->chi || !d->sigma_s || !d->speed) return MCDC_ERR_ARG;
  if (!d->surf_coef || !d->surf_bc || !d->cell_offset || !d->hs_surface || !d->hs_sense || !d->cell_material)
    return MCDC_ERR_ARG;
  if (!d->src_group_pdf || !d->time_edges || !d->census_times) return MCDC_ERR_ARG;
  if (d->n_time_bins < 1 || d->n_census < 1) return MCDC_ERR_GRID;
  const int G = d->n_groups, M = d->n_materials;
  for (int g = 0; g < G; ++g)
    if (!(d->speed[g] > 0.0) || !std::isfinite(d->speed[g])) return MCDC_ERR_XS;
  for (int m = 0; m < M; ++m) {
    bool fissile = false;
    double chi_sum = 0.0;
    for (int g = 0; g < G; ++g) {
      size_t mg = (size_t)m * G + g;
      double st = d->sigma_t[mg], sc = d->sigma_c[mg], sf = d->sigma_f[mg], nu = d->nu[mg];
      if (!(st >= 0.0) || !(sc >= 0.0) || !(sf >= 0.0) || !(nu >= 0.0) || !std::isfinite(st)) return MCDC_ERR_XS;
      if (nu >= 254.0) return MCDC_ERR_XS;
      double ss = 0.0;
      for (int gp = 0; gp < G; ++gp) {
        double v = d->sigma_s[mg * G + gp];
        if (!(v >= 0.0)) return MCDC_ERR_XS;
        ss += v;
      }
      if (std::fabs(st - (sc + ss + sf)) > 1e-12 * std::max(st, 1e-300) + 1e-300) return MCDC_ERR_XS;
      if (sf > 0.0) fissile = true;
      if (!(d->chi[mg] >= 0.0)) return MCDC_ERR_XS;
      chi_sum += d->chi[mg];
    }
    if (fissile && std::fabs(chi_sum - 1.0) > 1e-9) return MCDC_ERR_XS;
  }
  for (int s = 0; s < d->n_surfaces; ++s) {
    if (d->surf_bc[s] < 0 || d->surf_bc[s] > 2) return MCDC_ERR_GEOM;
    bool any = false;
    for (int i = 0; i < 9; ++i) {
      if (!std::isfinite(d->surf_coef[10 * s + i])) return MCDC_ERR_GEOM;
      if (d->surf_coef[10 * s + i] != 0.0) any = true;
    }
    if (!any || !std::isfinite(d->surf_coef[10 * s + 9])) return MCDC_ERR_GEOM;
  }
  if (d->cell_offset[0] != 0) return MCDC_ERR_GEOM;
  for (int c = 0; c < d->n_cells; ++c) {
    if (d->cell_offset[c + 1] <= d->cell_offset[c]) return MCDC_ERR_GEOM;
    if (d->cell_material[c] < 0 || d->cell_material[c] >= M) return MCDC_ERR_GEOM;
    for (int i = d->cell_offset[c]; i < d->cell_offset[c + 1]; ++i) {
      if (d->hs_surface[i] < 0 || d->hs_surface[i] >= d->n_surfaces) return MCDC_ERR_GEOM;
      if (d->hs_sense[i] != 1 && d->hs_sense[i] != -1) return MCDC_ERR_GEOM;
    }
  }
  double pdf_sum = 0.0;
  for (int g = 0; g < G; ++g) {
    if (!(d->src_group_pdf[g] >= 0.0)) return MCDC_ERR_ARG;
    pdf_sum += d->src_group_pdf[g];
  }
  if (std::fabs(pdf_sum - 1.0) > 1e-9) return MCDC_ERR_ARG;
  for (int a = 0; a < 3; ++a) {
    if (!(d->src_lo[a] <= d->src_hi[a]) || !std::isfinite(d->src_lo[a]) || !std::isfinite(d->src_hi[a])) return MCDC_ERR_ARG;
    if (d->mesh_n[a] < 1 || !(d->mesh_lo[a] < d->mesh_hi[a])) return MCDC_ERR_GRID;
    if (d->mesh_n[a] > 1 && (!std::isfinite(d->mesh_lo[a]) || !std::isfinite(d->mesh_hi[a]))) return MCDC_ERR_GRID;
  }
  if (d->src_dir_mode != MCDC_DIR_ISOTROPIC && d->src_dir_mode != MCDC_DIR_FIXED) return MCDC_ERR_ARG;
  if (d->src_dir_mode == MCDC_DIR_FIXED) {
    double n2 = d->src_dir[0] * d->src_dir[0] + d->src_dir[1] * d->src_dir[1] + d->src_dir[2] * d->src_dir[2];
    if (std::fabs(n2 - 1.0) > 1e-12) return MCDC_ERR_ARG;
  }
  if (!(d->src_t0 <= d->src_t1)) return MCDC_ERR_ARG;
  for (int i = 0; i < d->n_time_bins; ++i)
    if (!(d->time_edges[i] < d->time_edges[i + 1])) return MCDC_ERR_GRID;
  for (int k = 0; k < d->n_census; ++k) {
    if (!std::isfinite(d->census_times[k])) return MCDC_ERR_GRID;
    if (k > 0 && !(d->census_times[k - 1] < d->census_times[k])) return MCDC_ERR_GRID;
  }
  if (!(d->census_times[0] > d->src_t0) || !(d->src_t1 <= d->census_times[d->n_census - 1])) return MCDC_ERR_GRID;
  return MCDC_OK;
}

// ---------------------------------------------------------------------------------------------
// surface classification, cell boxes, neighbour tables, source locator grid
// ---------------------------------------------------------------------------------------------
void classify_surface(const double *c, int &type, double4 &q) {
  q = make_double4(0, 0, 0, 0);
  const bool quad = c[0] != 0 || c[1] != 0 || c[2] != 0 || c[3] != 0 || c[4] != 0 || c[5] != 0;
  if (!quad) {
    int nz = 0, ax = -1;
    for (int a = 0; a < 3; ++a)
      if (c[6 + a] != 0.0) { nz++; ax = a; }
    if (nz == 1) {
      type = ST_PLANE_X + ax;
      q.x = -c[9] / c[6 + ax];
      q.y = c[6 + ax] > 0.0 ? 1.0 : -1.0;
      return;
    }
    type = ST_QUADRIC;
    return;
  }
  if (c[0] == c[1] && c[0] != 0.0 && c[2] == 0 && c[3] == 0 && c[4] == 0 && c[5] == 0 && c[8] == 0) {
    double A = c[0];
    double x0 = -c[6] / (2.0 * A), y0 = -c[7] / (2.0 * A);
    double r2 = x0 * x0 + y0 * y0 - c[9] / A;
    if (r2 > 0.0) {
      type = ST_CYL_Z;
      q.x = x0; q.y = y0; q.z = r2; q.w = A > 0.0 ? 1.0 : -1.0;
      return;
    }
  }
  type = ST_QUADRIC;
}

Box cell_box(const mcdc_problem &P, const std::vector<int> &type, const std::vector<double4> &q, int c, bool pad = true) {
  Box b;
  for (int a = 0; a < 3; ++a) { b.lo[a] = -HINF; b.hi[a] = HINF; }
  if (!P.rgn_off.empty() && P.rgn_off[c] < P.rgn_off[c + 1]) return b;   // a general region: its half-spaces bound nothing
  for (int i = P.cell_off[c]; i < P.cell_off[c + 1]; ++i) {
    int s = P.hs_surface[i], sense = P.hs_sense[i];
    if (type[s] <= ST_PLANE_Z) {
      int a = type[s] - ST_PLANE_X;
      bool below = (q[s].y > 0.0) == (sense < 0);          // coordinate < position
      if (below) b.hi[a] = std::min(b.hi[a], q[s].x); else b.lo[a] = std::max(b.lo[a], q[s].x);
    } else if (type[s] == ST_CYL_Z && (double)sense * q[s].w < 0.0) {   // inside the cylinder
      double r = std::sqrt(q[s].z);
      b.lo[0] = std::max(b.lo[0], q[s].x - r); b.hi[0] = std::min(b.hi[0], q[s].x + r);
      b.lo[1] = std::max(b.lo[1], q[s].y - r); b.hi[1] = std::min(b.hi[1], q[s].y + r);
    }
  }
  for (int a = 0; a < 3 && pad; ++a) {                     // pad: a point within rounding of a face stays inside
    double ref = 1.0 + (std::isfinite(b.lo[a]) ? std::fabs(b.lo[a]) : 0.0) + (std::isfinite(b.hi[a]) ? std::fabs(b.hi[a]) : 0.0);
    b.lo[a] -= 1e-6 * ref; b.hi[a] += 1e-6 * ref;
  }
  return b;
}

inline bool boxes_touch(const Box &a, const Box &b) {
  for (int i = 0; i < 3; ++i)
    if (a.hi[i] < b.lo[i] || b.hi[i] < a.lo[i]) return false;
  return true;
}

}  // namespace

// =============================================================================================
// create / destroy / reset
// =============================================================================================
extern "C" int mcdc_problem_create(const mcdc_problem_desc *d, mcdc_problem **out) {
  return mcdc_problem_create_csg(d, nullptr, nullptr, out);
}

extern "C" int mcdc_problem_create_csg(const mcdc_problem_desc *d, const int32_t *region_offset, const int32_t *region_rpn,
                                       mcdc_problem **out) {
  if (!out) return MCDC_ERR_ARG;
  int rc = validate(d);
  if (rc != MCDC_OK) return rc;
  if ((region_offset == nullptr) != (region_rpn == nullptr)) return MCDC_ERR_ARG;
  if (region_offset) {                                    // Appendix J: well-formed postfix expressions only
    if (region_offset[0] != 0) return MCDC_ERR_GEOM;
    for (int c = 0; c < d->n_cells; ++c) {
      const int nh = d->cell_offset[c + 1] - d->cell_offset[c];
      if (region_offset[c + 1] < region_offset[c]) return MCDC_ERR_GEOM;
      int depth = 0;
      for (int k = region_offset[c]; k < region_offset[c + 1]; ++k) {
        const int t = region_rpn[k];
        if (t >= 0) { if (t >= nh) return MCDC_ERR_GEOM; if (++depth > 32) return MCDC_ERR_GEOM; }
        else if (t == MCDC_RGN_NOT) { if (depth < 1) return MCDC_ERR_GEOM; }
        else if (t == MCDC_RGN_AND || t == MCDC_RGN_OR) { if (depth < 2) return MCDC_ERR_GEOM; --depth; }
        else return MCDC_ERR_GEOM;
      }
      if (region_offset[c + 1] > region_offset[c] && depth != 1) return MCDC_ERR_GEOM;
    }
  }
  mcdc_problem *p = new (std::nothrow) mcdc_problem();
  if (!p) return MCDC_ERR_NOMEM;
  const int G = d->n_groups, M = d->n_materials, S = d->n_surfaces, C = d->n_cells;
  p->G = G; p->M = M; p->S = S; p->C = C; p->K = d->n_census; p->Nt = d->n_time_bins;
  const size_t MG = (size_t)M * G;
  p->sigma_t.assign(d->sigma_t, d->sigma_t + MG); p->sigma_c.assign(d->sigma_c, d->sigma_c + MG);
  p->sigma_f.assign(d->sigma_f, d->sigma_f + MG); p->nu.assign(d->nu, d->nu + MG);
  p->chi.assign(d->chi, d->chi + MG); p->sigma_s.assign(d->sigma_s, d->sigma_s + MG * G);
  p->speed.assign(d->speed, d->speed + G);
  p->surf_coef.assign(d->surf_coef, d->surf_coef + (size_t)10 * S);
  p->surf_bc.assign(d->surf_bc, d->surf_bc + S);
  p->cell_off.assign(d->cell_offset, d->cell_offset + C + 1);
  const int nhs = p->cell_off[C];
  p->hs_surface.assign(d->hs_surface, d->hs_surface + nhs);
  p->hs_sense.assign(d->hs_sense, d->hs_sense + nhs);
  p->cell_mat.assign(d->cell_material, d->cell_material + C);
  bool has_regions = false;
  if (region_offset && region_offset[C] > 0) {
    p->rgn_off.assign(region_offset, region_offset + C + 1);
    p->rgn_tok.assign(region_rpn, region_rpn + region_offset[C]);
    has_regions = true;
  }
  p->src_pdf.assign(d->src_group_pdf, d->src_group_pdf + G);
  p->T.assign(d->time_edges, d->time_edges + d->n_time_bins + 1);
  p->census.assign(d->census_times, d->census_times + d->n_census);
  for (int a = 0; a < 3; ++a) {
    p->src_lo[a] = d->src_lo[a]; p->src_hi[a] = d->src_hi[a]; p->src_dir[a] = d->src_dir[a];
    p->mesh_lo[a] = d->mesh_lo[a]; p->mesh_hi[a] = d->mesh_hi[a]; p->mesh_n[a] = d->mesh_n[a];
  }
  p->src_t0 = d->src_t0; p->src_t1 = d->src_t1; p->src_dir_mode = d->src_dir_mode;
  p->n_spatial = (size_t)d->mesh_n[0] * d->mesh_n[1] * d->mesh_n[2];
  p->n_bins = (size_t)p->Nt * G * p->n_spatial;

  // ---- derived cross-section tables (same summation order as the definition, A.1 / A.6) ----
  std::vector<double> inv_sig_t(MG), s_tot(MG), s_sc(MG), cdf_s(MG * G), cdf_chi(MG), inv_speed(G), src_cdf(G);
  std::vector<int> last_s(MG, 0), last_chi(M, 0);
  for (size_t mg = 0; mg < MG; ++mg) {
    double run = 0.0;
    for (int gp = 0; gp < G; ++gp) {
      double v = p->sigma_s[mg * G + gp];
      run += v;
      cdf_s[mg * G + gp] = run;
      if (v != 0.0) last_s[mg] = gp;
    }
    s_tot[mg] = run;
    s_sc[mg] = run + p->sigma_c[mg];
    inv_sig_t[mg] = p->sigma_t[mg] > 0.0 ? 1.0 / p->sigma_t[mg] : HINF;   // void: -log(xi) * inf = no collision (A.2)
  }
  for (int m = 0; m < M; ++m) {
    double run = 0.0;
    for (int g = 0; g < G; ++g) {
      double v = p->chi[(size_t)m * G + g];
      run += v;
      cdf_chi[(size_t)m * G + g] = run;
      if (v != 0.0) last_chi[m] = g;
    }
  }
  int src_last = 0;
  {
    double run = 0.0;
    for (int g = 0; g < G; ++g) {
      run += p->src_pdf[g];
      src_cdf[g] = run;
      if (p->src_pdf[g] != 0.0) src_last = g;
      inv_speed[g] = 1.0 / p->speed[g];
    }
  }
  // ---- geometry tables ----
  std::vector<int> type(S);
  std::vector<double4> q(S);
  for (int s = 0; s < S; ++s) classify_surface(&p->surf_coef[(size_t)10 * s], type[s], q[s]);
  std::vector<int> hs(nhs);
  for (int i = 0; i < nhs; ++i)
    hs[i] = (p->hs_surface[i] << 6) | (p->surf_bc[p->hs_surface[i]] << 4) | (type[p->hs_surface[i]] << 1) | (p->hs_sense[i] > 0 ? 1 : 0);
  std::vector<Box> box(C);
  for (int c = 0; c < C; ++c) box[c] = cell_box(*p, type, q, c);
  // cells listing half-space (s, sense): index 2*s + (sense>0)
  std::vector<std::vector<int>> users((size_t)2 * S);
  auto user_key = [&](int i) { return (size_t)2 * p->hs_surface[i] + (p->hs_sense[i] > 0 ? 1 : 0); };
  for (int c = 0; c < C; ++c)
    for (int i = p->cell_off[c]; i < p->cell_off[c + 1]; ++i) users[user_key(i)].push_back(c);
  std::vector<int> nb_off(nhs + 1, 0), nb_cell;
  for (int c = 0; c < C; ++c)
    for (int i = p->cell_off[c]; i < p->cell_off[c + 1]; ++i) {
      const std::vector<int> &cand = users[user_key(i) ^ 1];          // same surface, opposite sense
      for (int c2 : cand)
        if (c2 != c && boxes_touch(box[c], box[c2])) nb_cell.push_back(c2);  // increasing id by construction
      if (has_regions)                                                // under a NOT the listed sense says nothing
        for (int c2 : users[user_key(i)])
          if (c2 != c && boxes_touch(box[c], box[c2])) nb_cell.push_back(c2);
      nb_off[i + 1] = (int)nb_cell.size();
    }
  // ---- typed cells (mcdc_types.h): tightest axis-aligned plane per (axis, side) = face, the rest = other ----
  std::vector<std::array<double, 6>> bound(C);
  std::vector<std::array<int, 6>> face(C);
  std::vector<std::vector<int>> others(C);
  for (int c = 0; c < C; ++c) {
    for (int a = 0; a < 3; ++a) { bound[c][2 * a] = -HINF; bound[c][2 * a + 1] = HINF; face[c][2 * a] = face[c][2 * a + 1] = -1; }
    // (a general region has no faces: under OR / NOT a listed plane bounds nothing, so all its surfaces are "others")
    const bool is_region = has_regions && p->rgn_off[c] < p->rgn_off[c + 1];
    for (int i = p->cell_off[c]; i < p->cell_off[c + 1] && !is_region; ++i) {
      const int s = p->hs_surface[i];
      if (type[s] > ST_PLANE_Z) continue;
      const int a = type[s] - ST_PLANE_X;
      const bool below = (q[s].y > 0.0) == (p->hs_sense[i] < 0);          // coordinate < position
      const int f = 2 * a + (below ? 1 : 0);
      const bool tighter = below ? (q[s].x < bound[c][f]) : (q[s].x > bound[c][f]);
      if (tighter) { bound[c][f] = q[s].x; face[c][f] = i; }              // equal positions: the earlier slot stays
    }
    for (int i = p->cell_off[c]; i < p->cell_off[c + 1]; ++i) {
      bool is_face = false;
      for (int f = 0; f < 6; ++f) is_face = is_face || face[c][f] == i;
      if (!is_face) others[c].push_back(i);
    }
  }
  // candidate neighbours: the one sharing the largest part of the face first (cells do not overlap, so the order
  // of the tests cannot change which cell contains the point -- DESIGN.md section 2)
  {
    std::vector<Box> ubox(C);
    for (int c = 0; c < C; ++c) ubox[c] = cell_box(*p, type, q, c, false);
    auto overlap = [&](int c1, int c2) {
      double m = 1.0;
      int finite = 0;
      for (int a = 0; a < 3; ++a) {
        const double lo = std::max(ubox[c1].lo[a], ubox[c2].lo[a]), hi = std::min(ubox[c1].hi[a], ubox[c2].hi[a]);
        if (!std::isfinite(lo) || !std::isfinite(hi)) continue;
        const double w = hi - lo;
        if (w > 1e-9 * (1.0 + std::fabs(lo) + std::fabs(hi))) { m *= w; finite++; }   // skip the shared (zero-width) axis
        else if (w < -1e-9 * (1.0 + std::fabs(lo) + std::fabs(hi))) return -1.0;
      }
      return finite ? m : 0.0;
    };
    for (int c = 0; c < C; ++c)
      for (int i = p->cell_off[c]; i < p->cell_off[c + 1]; ++i)
        std::stable_sort(nb_cell.begin() + nb_off[i], nb_cell.begin() + nb_off[i + 1],
                         [&](int x, int y) { return overlap(c, x) > overlap(c, y); });
  }
  // the tally mesh covers the geometry and the time grid covers the run: the score needs no clipping
  int score_fast = 1;
  for (int c = 0; c < C && score_fast; ++c) {
    const Box b = cell_box(*p, type, q, c, false);
    for (int a = 0; a < 3; ++a)
      if (!(p->mesh_lo[a] <= b.lo[a]) || !(p->mesh_hi[a] >= b.hi[a])) score_fast = 0;
  }
  if (!(p->T[0] <= p->src_t0) || !(p->T[p->Nt] >= p->census[p->K - 1])) score_fast = 0;

  // ---- compact tables of k_warp (mcdc_types.h): certificates, one-bin cells, one-bin census intervals ----
  // "Certificates": at a transmission the new cell is found by A.5's search over the cells on the other side.  Where
  // geometry alone proves that ONE candidate n holds every point of the crossed surface patch, the kernel may take n
  // without testing.  The patch of half-space (s, sense) of cell c lies inside R = c's bounding box (flattened onto the
  // plane, or cut to the cylinder's bounding box).  n is certified when (1) it lists s with the opposite sense -- as its
  // own face at the same position when s is a plane; (2) on every other axis n's plane bounds enclose R, where a bound
  // that R takes from one of c's own planes may coincide (the kernel then requires the point to lie strictly inside c's
  // forward faces) and any other bound must clear R by a margin; (3) each of n's remaining half-spaces holds on all of R
  // by a margin (axis-aligned planes and z-cylinders only; a general quadric is never certified).  Cells do not overlap
  // (header), so no other cell can hold such a point.  Points that fail the kernel's strict test take the full search.
  std::vector<Box> ubox(C);
  for (int c = 0; c < C; ++c) ubox[c] = cell_box(*p, type, q, c, false);
  auto holds_on_box = [&](int t, int sense, const Box &R) -> bool {
    if (type[t] <= ST_PLANE_Z) {
      const int a = type[t] - ST_PLANE_X;
      const double pos = q[t].x, m = 1e-9 * (1.0 + std::fabs(pos));
      const bool below = (q[t].y > 0.0) == (sense < 0);                     // coordinate < position required
      return below ? (R.hi[a] < pos - m) : (R.lo[a] > pos + m);
    }
    if (type[t] == ST_CYL_Z) {
      const bool inside = (double)sense * q[t].w < 0.0;
      const double x0 = q[t].x, y0 = q[t].y, r2 = q[t].z;
      const double dxn = std::max(0.0, std::max(R.lo[0] - x0, x0 - R.hi[0])), dyn = std::max(0.0, std::max(R.lo[1] - y0, y0 - R.hi[1]));
      const double dxx = std::max(std::fabs(R.lo[0] - x0), std::fabs(R.hi[0] - x0)), dyx = std::max(std::fabs(R.lo[1] - y0), std::fabs(R.hi[1] - y0));
      return inside ? (dxx * dxx + dyx * dyx < r2 * (1.0 - 1e-9)) : (dxn * dxn + dyn * dyn > r2 * (1.0 + 1e-9));
    }
    return false;
  };
  auto encloses = [&](int n, int c, const Box &R, int skip_axis) -> bool {   // condition (2)
    for (int b = 0; b < 3; ++b) {
      if (b == skip_axis) continue;
      const double m = 1e-9 * (1.0 + (std::isfinite(R.lo[b]) ? std::fabs(R.lo[b]) : 0.0) + (std::isfinite(R.hi[b]) ? std::fabs(R.hi[b]) : 0.0));
      const bool lo_ok = bound[n][2 * b] <= bound[c][2 * b] || bound[n][2 * b] < R.lo[b] - m;
      const bool hi_ok = bound[n][2 * b + 1] >= bound[c][2 * b + 1] || bound[n][2 * b + 1] > R.hi[b] + m;
      if (!lo_ok || !hi_ok) return false;
    }
    return true;
  };
  auto region_cell = [&](int c) { return has_regions && p->rgn_off[c] < p->rgn_off[c + 1]; };
  auto certified = [&](int c, int i) -> int {                                // neighbour across half-space slot i of cell c
    const int s = p->hs_surface[i];
    if (p->surf_bc[s] != MCDC_BC_TRANSMISSION) return -1;
    if (region_cell(c)) return -1;                                           // its surface patches are not bounded by its box
    Box R = ubox[c];
    int axis = -1, f = -1;
    if (type[s] <= ST_PLANE_Z) {
      axis = type[s] - ST_PLANE_X;
      for (int k = 0; k < 2; ++k)
        if (face[c][2 * axis + k] == i) f = 2 * axis + k;
      if (f < 0) return -1;                                                   // a redundant plane: never the nearest one
      R.lo[axis] = R.hi[axis] = bound[c][f];
    } else if (type[s] == ST_CYL_Z) {
      const double r = std::sqrt(q[s].z);
      R.lo[0] = std::max(R.lo[0], q[s].x - r); R.hi[0] = std::min(R.hi[0], q[s].x + r);
      R.lo[1] = std::max(R.lo[1], q[s].y - r); R.hi[1] = std::min(R.hi[1], q[s].y + r);
    } else return -1;
    for (int k = nb_off[i]; k < nb_off[i + 1]; ++k) {
      const int n = nb_cell[k];
      if (region_cell(n)) continue;                                          // membership of a region is never proved here
      if (axis >= 0) {
        const int fo = f ^ 1;
        if (face[n][fo] < 0 || p->hs_surface[face[n][fo]] != s) continue;
      }
      if (!encloses(n, c, R, axis)) continue;
      bool ok = true;
      for (int o : others[n]) {
        if (p->hs_surface[o] == s) continue;
        ok = ok && holds_on_box(p->hs_surface[o], p->hs_sense[o], R);
      }
      if (ok) return n;
    }
    return -1;
  };
  bool warp_ok = S + 2 < (int)NONE16 && C < (int)NONE16 && M <= 255 && G <= 254 && p->K <= 4095;
  std::vector<unsigned char> cell2((size_t)C * CELL2_BYTES, 0), other2;
  size_t n_cert = 0, n_transm = 0;
  for (int c = 0; c < C && warp_ok; ++c) {
    unsigned char *r = cell2.data() + (size_t)c * CELL2_BYTES;
    if (p->cell_off[c + 1] - p->cell_off[c] > 255 || others[c].size() > 255 || other2.size() / OTHER2_BYTES > 65000) { warp_ok = false; break; }
    uint16_t fs[6], fn[6], fbc = 0;
    uint8_t fi[6];
    for (int f = 0; f < 6; ++f) {
      // a side without a face names one of the two sentinel entries behind the surface table: position +inf (upper
      // side) or -inf (lower side), so that the kernel reads every face position without a test
      fs[f] = (uint16_t)(S + ((f & 1) ? 0 : 1)); fn[f] = (uint16_t)NONE16; fi[f] = 0;
      const int i = face[c][f];
      if (i < 0) continue;
      const int s = p->hs_surface[i];
      fs[f] = (uint16_t)s; fi[f] = (uint8_t)(i - p->cell_off[c]);
      fbc |= (uint16_t)(p->surf_bc[s] << (2 * f));
      const int n = certified(c, i);
      if (p->surf_bc[s] == MCDC_BC_TRANSMISSION) { n_transm++; if (n >= 0) n_cert++; }
      if (n >= 0) fn[f] = (uint16_t)n;
    }
    std::memcpy(r + C2_FACE_SURF, fs, 12); std::memcpy(r + C2_FACE_NB, fn, 12); std::memcpy(r + C2_FACE_IDX, fi, 6);
    std::memcpy(r + C2_FACE_BC, &fbc, 2);
    const uint32_t info = (uint32_t)others[c].size() | ((uint32_t)p->cell_mat[c] << 8) | ((uint32_t)(other2.size() / OTHER2_BYTES) << 16);
    std::memcpy(r + C2_INFO, &info, 4);
    for (int i : others[c]) {
      const int s = p->hs_surface[i];
      const int n = certified(c, i);
      if (p->surf_bc[s] == MCDC_BC_TRANSMISSION) { n_transm++; if (n >= 0) n_cert++; }
      const uint32_t w0 = (uint32_t)s | ((uint32_t)(n >= 0 ? n : (int)NONE16) << 16);
      const uint32_t flags = (p->hs_sense[i] > 0 ? 1u : 0u) | ((uint32_t)type[s] << 1) | ((uint32_t)p->surf_bc[s] << 4);
      const uint32_t w1 = (uint32_t)(i - p->cell_off[c]) | (flags << 8);
      unsigned char e[8];
      std::memcpy(e, &w0, 4); std::memcpy(e + 4, &w1, 4);
      other2.insert(other2.end(), e, e + 8);
    }
    // the one spatial tally bin that holds the whole cell (the score is then a single addition)
    uint32_t cbin = NONE32;
    if (score_fast) {
      int idx[3] = {0, 0, 0};
      bool one = true;
      for (int a = 0; a < 3 && one; ++a) {
        if (p->mesh_n[a] == 1) continue;
        const double d = (p->mesh_hi[a] - p->mesh_lo[a]) / p->mesh_n[a];
        const double lo = ubox[c].lo[a], hi = ubox[c].hi[a];
        if (!std::isfinite(lo) || !std::isfinite(hi)) { one = false; break; }
        const double tol = 1e-12 * (1.0 + std::fabs(lo) + std::fabs(hi)) / d;
        const double i_lo = std::floor((lo - p->mesh_lo[a]) / d + tol), i_hi = std::ceil((hi - p->mesh_lo[a]) / d - tol) - 1.0;
        if (i_lo != i_hi || i_lo < 0.0 || i_lo > (double)(p->mesh_n[a] - 1)) one = false; else idx[a] = (int)i_lo;
      }
      if (one) cbin = (uint32_t)((idx[2] * p->mesh_n[1] + idx[1]) * p->mesh_n[0] + idx[0]);
    }
    std::memcpy(r + C2_BIN, &cbin, 4);
    if (cbin != NONE32) p->n_one_bin++;
  }
  if (other2.empty()) other2.resize(OTHER2_BYTES, 0);
  p->n_cert = n_cert; p->n_transm = n_transm;
  // census interval k = (C[k-1] (or the source start), C[k]]: the time bin that holds all of it, if one does
  std::vector<int> tbin_k(p->K, -1), it0_k(p->K, 0);
  for (int k = 0; k < p->K; ++k) {
    const double a_k = (k == 0) ? p->src_t0 : p->census[k - 1];
    int j = 0;
    for (int i = 0; i < p->Nt; ++i)
      if (p->T[i] <= a_k) j = i;
    it0_k[k] = j;
    if (score_fast && p->T[j] <= a_k && p->census[k] <= p->T[j + 1]) tbin_k[k] = j;
  }

  // ---- source locator grid ----
  int loc_n[3];
  double loc_lo[3], loc_inv_d[3];
  for (int a = 0; a < 3; ++a) {
    double ext = p->src_hi[a] - p->src_lo[a];
    loc_n[a] = ext > 0.0 ? 16 : 1;
    loc_lo[a] = p->src_lo[a];
    loc_inv_d[a] = ext > 0.0 ? loc_n[a] / ext : 0.0;
  }
  const int nvox = loc_n[0] * loc_n[1] * loc_n[2];
  std::vector<int> loc_off(nvox + 1, 0), loc_cell;
  for (int vz = 0; vz < loc_n[2]; ++vz)
    for (int vy = 0; vy < loc_n[1]; ++vy)
      for (int vx = 0; vx < loc_n[0]; ++vx) {
        int v[3] = {vx, vy, vz};
        Box vb;
        for (int a = 0; a < 3; ++a) {
          double ext = p->src_hi[a] - p->src_lo[a];
          double dlt = ext / loc_n[a];
          vb.lo[a] = p->src_lo[a] + v[a] * dlt - 1e-9 * (1.0 + std::fabs(p->src_lo[a]) + ext);
          vb.hi[a] = p->src_lo[a] + (v[a] + 1) * dlt + 1e-9 * (1.0 + std::fabs(p->src_lo[a]) + ext);
        }
        for (int c = 0; c < C; ++c)
          if (boxes_touch(vb, box[c])) loc_cell.push_back(c);
        loc_off[(vz * loc_n[1] + vy) * loc_n[0] + vx + 1] = (int)loc_cell.size();
      }

  // ---- upload ----
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { delete p; return MCDC_ERR_CUDA; }
  int n_sm = 0;                                          // (one attribute: cudaGetDeviceProperties costs ~1 ms)
  if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm <= 0) { delete p; return MCDC_ERR_CUDA; }
  p->n_sm = n_sm;
  Tables &t = p->tab;
  DeviceArena &ar = p->arena;
  t.G = G; t.M = M; t.S = S; t.C = C; t.K = p->K; t.Nt = p->Nt;
  // one blob, 16-byte aligned pieces, hot tables first
  std::vector<unsigned char> blob;
  auto put = [&](const void *src, size_t bytes) -> uint32_t {
    size_t off = (blob.size() + 15) / 16 * 16;
    blob.resize(off + std::max<size_t>(bytes, 16), 0);
    if (bytes) std::memcpy(blob.data() + off, src, bytes);
    return (uint32_t)off;
  };
  auto putd = [&](const std::vector<double> &v) { return put(v.data(), v.size() * sizeof(double)); };
  auto puti = [&](const std::vector<int> &v) { return put(v.data(), v.size() * sizeof(int)); };
  t.o_sig_t = putd(p->sigma_t); t.o_inv_sig_t = putd(inv_sig_t); t.o_sig_s_tot = putd(s_tot); t.o_sig_sc = putd(s_sc);
  t.o_sig_f = putd(p->sigma_f); t.o_nu = putd(p->nu); t.o_cdf_s = putd(cdf_s); t.o_last_s = puti(last_s);
  t.o_cdf_chi = putd(cdf_chi); t.o_last_chi = puti(last_chi); t.o_speed = putd(p->speed); t.o_inv_speed = putd(inv_speed);
  t.o_T = putd(p->T); t.o_census = putd(p->census); t.o_src_cdf = putd(src_cdf);
  {
    std::vector<double> cap_frac((size_t)M * G);          // Sigma_c / Sigma_t (implicit capture, Appendix G.1)
    for (size_t i = 0; i < cap_frac.size(); ++i) cap_frac[i] = p->sigma_t[i] > 0.0 ? p->sigma_c[i] / p->sigma_t[i] : 0.0;
    t.o_cap_frac = putd(cap_frac);
  }
  t.implicit_capture = 0; t.wr_threshold = 0.0; t.wr_survive = 0.0;
  t.o_tbin_k = puti(tbin_k); t.o_it0_k = puti(it0_k);
  {                                                      // + the two sentinel positions of sides without a face
    std::vector<double4> qs(q);
    qs.push_back(make_double4(HINF, 0.0, 0.0, 0.0)); qs.push_back(make_double4(-HINF, 0.0, 0.0, 0.0));
    t.o_surf_q = put(qs.data(), qs.size() * sizeof(double4));
  }
  t.o_cell2 = put(cell2.data(), cell2.size()); t.o_other2 = put(other2.data(), other2.size());
  bool any_quadric = false;
  for (int s = 0; s < S; ++s) any_quadric = any_quadric || type[s] == ST_QUADRIC;
  // everything above is the hot prefix k_warp stages in shared memory; the generic tables below stay in L2
  const size_t hot = (blob.size() + 15) / 16 * 16;
  t.o_surf_bc = puti(p->surf_bc); t.o_cell_off = puti(p->cell_off); t.o_hs = puti(hs); t.o_cell_mat = puti(p->cell_mat);
  t.o_nb_off = puti(nb_off); t.o_nb_cell = puti(nb_cell);
  t.o_loc_off = puti(loc_off); t.o_loc_cell = puti(loc_cell);
  t.o_surf_coef = putd(p->surf_coef);
  t.has_regions = has_regions ? 1 : 0;
  t.o_rgn_off = 0; t.o_rgn_tok = 0;
  if (has_regions) { t.o_rgn_off = puti(p->rgn_off); t.o_rgn_tok = puti(p->rgn_tok); }
  t.score_fast = score_fast;
  t.warp_ok = warp_ok ? 1 : 0;
  {
    bool all1 = p->n_one_bin == (size_t)C;
    for (int k = 0; k < p->K; ++k) all1 = all1 && tbin_k[k] >= 0;
    t.all_one_bin = all1 ? 1 : 0;
  }
  (void)any_quadric;
  blob.resize((blob.size() + 15) / 16 * 16, 0);
  t.hot_bytes = (uint32_t)hot;
  t.blob = ar.upload(blob);
  t.src_last = src_last; t.src_dir_mode = p->src_dir_mode;
  // A point source that lies strictly inside exactly one cell (every half-space of the cell holds with a margin, so
  // the on-surface direction rule of A.3 cannot come into play) needs no per-particle cell search.
  t.src_cell = -1;
  if (!has_regions && p->src_lo[0] == p->src_hi[0] && p->src_lo[1] == p->src_hi[1] && p->src_lo[2] == p->src_hi[2]) {
    const double x = p->src_lo[0], y = p->src_lo[1], z = p->src_lo[2];
    int found = -1, n_found = 0;
    bool near_surface = false;
    for (int c = 0; c < C; ++c) {
      bool inside = true;
      for (int i = p->cell_off[c]; i < p->cell_off[c + 1] && inside; ++i) {
        const double *k = &p->surf_coef[(size_t)10 * p->hs_surface[i]];
        const double terms[10] = {k[0] * x * x, k[1] * y * y, k[2] * z * z, k[3] * x * y, k[4] * x * z, k[5] * y * z,
                                  k[6] * x, k[7] * y, k[8] * z, k[9]};
        double f = 0.0, mag = 0.0;
        for (int j = 0; j < 10; ++j) { f += terms[j]; mag += std::fabs(terms[j]); }
        if (std::fabs(f) <= 1e-9 * (mag + 1e-300)) { near_surface = true; inside = false; }
        else if ((f > 0.0) != (p->hs_sense[i] > 0)) inside = false;
      }
      if (inside) { found = c; ++n_found; }
    }
    if (!near_surface && n_found == 1) t.src_cell = found;
  }
  t.src_chk = 0;
  for (int a = 0; a < 3; ++a) { t.src_clo[a] = -HINF; t.src_chi[a] = HINF; }
  if (t.src_cell < 0 && !has_regions) {
    // A source box inside the closure of ONE cell bounded by axis-aligned planes only: a particle drawn strictly inside
    // that cell's bounds is in it (a draw that rounds onto a face still takes the search, where the direction decides)
    for (int c = 0; c < C && t.src_cell < 0; ++c) {
      bool planes_only = p->cell_off[c + 1] > p->cell_off[c];
      for (int i = p->cell_off[c]; i < p->cell_off[c + 1]; ++i) planes_only = planes_only && type[p->hs_surface[i]] <= ST_PLANE_Z;
      if (!planes_only) continue;
      const Box b = cell_box(*p, type, q, c, false);
      bool inside = true;
      for (int a = 0; a < 3; ++a) inside = inside && p->src_lo[a] >= b.lo[a] && p->src_hi[a] <= b.hi[a];
      if (!inside) continue;
      t.src_cell = c; t.src_chk = 1;
      for (int a = 0; a < 3; ++a) { t.src_clo[a] = b.lo[a]; t.src_chi[a] = b.hi[a]; }
    }
  }
  t.src_t0 = p->src_t0; t.src_t1 = p->src_t1;
  for (int a = 0; a < 3; ++a) {
    t.src_lo[a] = p->src_lo[a]; t.src_hi[a] = p->src_hi[a]; t.src_dir[a] = p->src_dir[a];
    t.loc_n[a] = loc_n[a]; t.loc_lo[a] = loc_lo[a]; t.loc_inv_d[a] = loc_inv_d[a];
    t.mesh_lo[a] = p->mesh_lo[a]; t.mesh_hi[a] = p->mesh_hi[a]; t.mesh_n[a] = p->mesh_n[a];
    t.mesh_d[a] = (p->mesh_hi[a] - p->mesh_lo[a]) / (double)p->mesh_n[a];
    t.mesh_inv_d[a] = (p->mesh_n[a] > 1) ? 1.0 / t.mesh_d[a] : 0.0;
  }
  t.n_bins = p->n_bins;
  {
    Tables *dT = ar.zeros<Tables>(1);
    t.self_dev = dT;
    if (dT && cudaMemcpy(dT, &t, sizeof(Tables), cudaMemcpyHostToDevice) != cudaSuccess) ar.err = cudaErrorUnknown;
  }
  {
    // every accumulator of the handle in ONE zeroed allocation (each cudaMalloc + cudaMemset pair costs ~0.1 ms);
    // the counters the kernels poll or hit with atomics (ledger, queue cursors, source cursor) get 256 bytes each
    const size_t nb = p->n_bins, K = (size_t)p->K;
    auto up32 = [](size_t w) { return (w + 31) / 32 * 32; };               // 8-byte words, rounded to 256 bytes
    const size_t words = up32(2 * nb) + up32(4 * K) + up32((sizeof(DevCounters) + 7) / 8) + 32 + 32;
    unsigned long long *blk = ar.zeros<unsigned long long>(words);
    if (blk) {
      size_t o = 0;
      p->d_sum = (double *)(blk + o); o += nb;
      p->d_sumsq = (double *)(blk + o); o = up32(2 * nb);
      p->d_pop_w = (double *)(blk + o); p->d_pop_n = blk + o + K;
      p->d_pop_w_after = (double *)(blk + o + 2 * K); p->d_pop_n_after = blk + o + 3 * K; o += up32(4 * K);
      p->d_cnt = (DevCounters *)(blk + o); o += up32((sizeof(DevCounters) + 7) / 8);
      p->d_head_tail = blk + o; o += 32;
      p->d_hist_cursor = (uint32_t *)(blk + o); o += 32;
    }
  }
  if (ar.err != cudaSuccess) {
    ar.release();
    delete p;
    return MCDC_ERR_CUDA;
  }
  int occ = 1;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_transport, TRANSPORT_THREADS, 0) == cudaSuccess && occ > 0)
    p->blocks_per_sm = occ;
  *out = p;
  return MCDC_OK;
}

extern "C" void mcdc_problem_destroy(mcdc_problem *p) {
  if (!p) return;
  p->arena.release();
  for (auto &pr : p->ev_pairs) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
  for (cudaEvent_t e : {p->e_run0, p->e_run1, p->e_tr0, p->e_tr1})
    if (e) cudaEventDestroy(e);
  if (p->e_poll) cudaEventDestroy(p->e_poll);
  if (p->h_poll) cudaFreeHost(p->h_poll);
  if (p->d_ev) cudaFree(p->d_ev);
  if (p->d_xc_acc) cudaFree(p->d_xc_acc);
  if (p->d_sumc) cudaFree(p->d_sumc);
  if (p->d_sumsqc) cudaFree(p->d_sumsqc);
  delete p;
}

extern "C" int mcdc_problem_reset(mcdc_problem *p) {
  if (!p) return MCDC_ERR_ARG;
  CK(cudaMemsetAsync(p->d_sum, 0, p->n_bins * sizeof(double), p->stream));
  CK(cudaMemsetAsync(p->d_sumsq, 0, p->n_bins * sizeof(double), p->stream));
  CK(cudaMemsetAsync(p->d_pop_w, 0, p->K * sizeof(double), p->stream));
  CK(cudaMemsetAsync(p->d_pop_n, 0, p->K * sizeof(unsigned long long), p->stream));
  CK(cudaMemsetAsync(p->d_pop_w_after, 0, p->K * sizeof(double), p->stream));
  CK(cudaMemsetAsync(p->d_pop_n_after, 0, p->K * sizeof(unsigned long long), p->stream));
  CK(cudaMemsetAsync(p->d_cnt, 0, sizeof(DevCounters), p->stream));
  if (p->x_acc) CK(cudaMemsetAsync(p->x_acc, 0, (size_t)p->ws_slots * p->n_bins * sizeof(double), p->stream));
  if (p->d_xc_acc) {
    CK(cudaMemsetAsync(p->d_xc_acc, 0, (size_t)p->xc_slots * p->n_bins * sizeof(double), p->stream));
    CK(cudaMemsetAsync(p->d_sumc, 0, p->n_bins * sizeof(double), p->stream));
    CK(cudaMemsetAsync(p->d_sumsqc, 0, p->n_bins * sizeof(double), p->stream));
  }
  CK(cudaStreamSynchronize(p->stream));
  p->histories = p->batches = p->batch_size = p->launches = 0;
  p->ms_run = p->ms_transport = 0.0;
  p->ev_n = 0;
  return MCDC_OK;
}

// =============================================================================================
// workspace
// =============================================================================================
namespace {

// bank records: full = x y z ux uy uz t w, key, meta, hid = 92 B; birth = x y z t w, key, meta, hid = 68 B

struct WsLayout {
  size_t total = 0;
  size_t x_acc = 0, counts = 0, bank[4] = {0, 0, 0, 0};
  size_t q_flag = 0, q_data = 0;
  uint64_t q_cap = 0;
  size_t fixed = 0;          // bytes zeroed at bind (accumulators, counts, queue flags)
};

// slots * cap particles per bank; two full banks (live, census) and two birth banks (fission ping-pong)
uint64_t queue_capacity(uint64_t hist) {               // power of two, 2^20 .. 2^25 entries
  uint64_t c = 1ull << 20;
  while (c < hist && c < (1ull << 25)) c <<= 1;
  return c;
}

WsLayout layout(const mcdc_problem *p, uint32_t slots, uint64_t cap, uint64_t hist) {
  WsLayout L;
  size_t off = 0;
  L.x_acc = off; off += align_up((size_t)slots * p->n_bins * sizeof(double), 256);
  L.counts = off; off += align_up((size_t)10 * slots * sizeof(uint32_t), 256);   // 8 bank counters + one u64 (wfix) per slot
  L.q_cap = queue_capacity(hist);
  L.q_flag = off; off += align_up((size_t)L.q_cap * sizeof(uint32_t), 256);
  L.fixed = off;
  L.q_data = off; off += (size_t)6 * align_up((size_t)L.q_cap * 8, 256) + align_up((size_t)L.q_cap * 16, 256);
  const size_t n = (size_t)slots * cap;
  for (int b = 0; b < 4; ++b) {
    L.bank[b] = off;
    const int n_dbl = (b < 2) ? 8 : 5;
    off += (size_t)n_dbl * align_up(n * 8, 256) + align_up(n * 8, 256) + align_up(n * 16, 256) + align_up(n * 4, 256);
  }
  L.total = off;
  return L;
}

void carve_bank(Bank &B, char *base, size_t off, size_t n, bool full, uint32_t *count, uint32_t *cursor) {
  char *q = base + off;
  auto take = [&](size_t bytes) { char *r = q; q += align_up(bytes, 256); return r; };
  B.x = (double *)take(n * 8); B.y = (double *)take(n * 8); B.z = (double *)take(n * 8);
  if (full) { B.ux = (double *)take(n * 8); B.uy = (double *)take(n * 8); B.uz = (double *)take(n * 8); }
  else B.ux = B.uy = B.uz = nullptr;
  B.t = (double *)take(n * 8); B.w = (double *)take(n * 8);
  B.key = (unsigned long long *)take(n * 8);
  B.meta = (int4 *)take(n * 16);
  B.hid = (uint32_t *)take(n * 4);
  B.count = count; B.cursor = cursor;
}

uint64_t default_cap(uint64_t hist, uint32_t slots) {
  uint64_t hb = (hist + slots - 1) / slots;
  return align_up((size_t)(2 * hb + 1024), 32);
}

}  // namespace

extern "C" int mcdc_workspace_size(const mcdc_problem *p, uint64_t max_hist, uint32_t max_slots, size_t *bytes) {
  if (!p || !bytes || max_hist == 0 || max_slots == 0 || max_hist > 0xFFFFFFF0ull) return MCDC_ERR_ARG;
  *bytes = layout(p, max_slots, default_cap(max_hist, max_slots), max_hist).total;
  return MCDC_OK;
}

extern "C" int mcdc_workspace_size_async(const mcdc_problem *p, uint64_t max_hist, uint32_t max_slots, size_t *bytes) {
  if (!p || !bytes || max_hist == 0 || max_slots == 0 || max_hist > 0xFFFFFFF0ull) return MCDC_ERR_ARG;
  *bytes = layout(p, max_slots, 0, max_hist).total;      // no particle banks: accumulators and the fission queue only
  return MCDC_OK;
}

extern "C" int mcdc_workspace_bind(mcdc_problem *p, void *dev_ptr, size_t bytes, uint64_t max_hist, uint32_t max_slots,
                                   void *cuda_stream) {
  if (!p || !dev_ptr || max_hist == 0 || max_slots == 0 || max_hist > 0xFFFFFFF0ull) return MCDC_ERR_ARG;
  if (((uintptr_t)dev_ptr & 255u) != 0) return MCDC_ERR_ARG;
  uint64_t cap = default_cap(max_hist, max_slots);
  WsLayout L = layout(p, max_slots, cap, max_hist);
  if (bytes < L.total) {                                  // enough for the asynchronous scheduler alone?
    cap = 0;
    L = layout(p, max_slots, 0, max_hist);
    if (bytes < L.total) return MCDC_ERR_NO_WORKSPACE;
  } else {
    // a larger workspace buys larger banks: grow cap while it fits
    uint64_t lo = cap, hi = cap * 64;
    while (lo + 32 <= hi) {
      uint64_t mid = align_up((size_t)((lo + hi) / 2), 32);
      if (mid * max_slots <= 0xFFFFFFF0ull && layout(p, max_slots, mid, max_hist).total <= bytes) lo = mid; else hi = mid - 32;
    }
    cap = lo;
    L = layout(p, max_slots, cap, max_hist);
  }
  p->ws = (char *)dev_ptr; p->ws_bytes = bytes; p->ws_hist = max_hist; p->ws_slots = max_slots;
  p->cap = (uint32_t)cap;
  p->stream = (cudaStream_t)cuda_stream;
  p->x_acc = (double *)(p->ws + L.x_acc);
  uint32_t *cnt = (uint32_t *)(p->ws + L.counts);
  p->counts_dev = cnt;
  {
    char *qd = p->ws + L.q_data;
    auto take = [&](size_t bytes) { char *r = qd; qd += align_up(bytes, 256); return r; };
    FissionQueue &Q = p->queue;
    Q.x = (double *)take(L.q_cap * 8); Q.y = (double *)take(L.q_cap * 8); Q.z = (double *)take(L.q_cap * 8);
    Q.t = (double *)take(L.q_cap * 8); Q.w = (double *)take(L.q_cap * 8);
    Q.key = (unsigned long long *)take(L.q_cap * 8);
    Q.meta = (int4 *)take(L.q_cap * 16);
    Q.flag = (uint32_t *)(p->ws + L.q_flag);
    Q.mask = (uint32_t)(L.q_cap - 1);
    Q.head_tail = p->d_head_tail;
  }
  CK(cudaMemsetAsync(p->d_head_tail, 0, 2 * sizeof(unsigned long long), (cudaStream_t)cuda_stream));
  const size_t n = (size_t)max_slots * cap;
  carve_bank(p->bankA, p->ws, L.bank[0], n, true, cnt + 0 * max_slots, cnt + 1 * max_slots);
  carve_bank(p->bankB, p->ws, L.bank[1], n, true, cnt + 2 * max_slots, cnt + 3 * max_slots);
  carve_bank(p->bankS1, p->ws, L.bank[2], n, false, cnt + 4 * max_slots, cnt + 5 * max_slots);
  carve_bank(p->bankS2, p->ws, L.bank[3], n, false, cnt + 6 * max_slots, cnt + 7 * max_slots);
  p->d_wfix = reinterpret_cast<unsigned long long *>(cnt + 8 * max_slots);
  CK(cudaMemsetAsync(p->ws, 0, L.fixed, p->stream));
  CK(cudaStreamSynchronize(p->stream));
  return MCDC_OK;
}

// =============================================================================================
// run
// =============================================================================================
namespace {

constexpr int SLAB_MAX_BINS = 8192;   // 64 KB of shared memory for the privatised tally slab

int step_of(const mcdc_problem *p, double t) {          // smallest k with C[k] > t, else K-1
  for (int k = 0; k < p->K; ++k)
    if (p->census[k] > t) return k;
  return p->K - 1;
}

struct SubBatch {
  uint64_t first_local;   // index of its first history within the run
  uint32_t n_hist;
  uint32_t n_slots;
  uint32_t hs;            // histories per slot
  int closeout;           // 0 none, 1 per-slot batches, 2 all slots form one batch
  uint32_t closeout_slots;   // slots the close-out covers (>= n_slots: earlier pieces of a split batch may have used more)
};

int run_subbatch(mcdc_problem *p, const SubBatch &sb, uint64_t seed, uint64_t first_history_id, bool record) {
  cudaEvent_t ev0 = p->e_tr0, ev1 = p->e_tr1;
  const uint32_t ns = sb.n_slots;
  const uint32_t ws_ns = p->ws_slots;
  uint32_t *counts_dev = p->counts_dev;
  std::vector<uint32_t> h_counts((size_t)8 * ws_ns);
  CK(cudaMemsetAsync(counts_dev, 0, (size_t)8 * ws_ns * sizeof(uint32_t), p->stream));
  Bank A = p->bankA, Bk = p->bankB, S1 = p->bankS1, S2 = p->bankS2;
  const int k_first = step_of(p, p->src_t0), k_last = step_of(p, p->src_t1);
  const size_t n_spatial_g = p->n_spatial * (size_t)p->G;
  TransportArgs ta;
  ta.x_acc = p->x_acc; ta.xc_acc = p->col_on ? p->d_xc_acc : nullptr; ta.cnt = p->d_cnt; ta.pop_w = p->d_pop_w; ta.pop_n = p->d_pop_n;
  ta.ev = record ? p->d_ev + (size_t)sb.first_local * 4 : nullptr;
  const int max_grid = p->n_sm * p->blocks_per_sm;
  uint64_t live_total = 0;

  for (int k = 0; k < p->K; ++k) {
    if (k >= k_first && k <= k_last) {
      SourceParams sp;
      sp.seed_mixed = mix64(seed + MCDC_GAMMA);
      sp.first_history = first_history_id + sb.first_local;
      sp.n_hist = sb.n_hist; sp.hb = sb.hs; sp.cap = p->cap; sp.k = k; sp.single_step = (k_first == k_last);
      k_source<<<(sb.n_hist + 255) / 256, 256, 0, p->stream>>>(p->tab, sp, A, p->d_cnt);
      p->launches++;
      live_total += sb.n_hist;          // upper bound, refined by the read-back below
    } else if (live_total == 0) {
      if (k > k_last) break;            // nothing alive and no source left
      continue;
    }
    StepParams st;
    st.k = k; st.is_last = (k == p->K - 1); st.t_census = p->census[k];
    {
      const double t_lo = (k == 0) ? p->src_t0 : p->census[k - 1];
      int it_lo = 0, it_hi = 0;
      for (int j = 0; j < p->Nt; ++j) {
        if (p->T[j] <= t_lo) it_lo = j;
        if (p->T[j] < p->census[k]) it_hi = j;
      }
      if (it_hi < it_lo) it_hi = it_lo;
      st.it_lo = it_lo; st.it_n = it_hi - it_lo + 1;
      size_t bins = (size_t)st.it_n * n_spatial_g;
      st.slab_bins = bins <= (size_t)SLAB_MAX_BINS ? (int)bins : 0;
    }
    st.n_slots = (int)ns; st.cap = p->cap; st.hb = sb.hs; st.record_events = record ? 1 : 0;
    const size_t smem = (size_t)st.slab_bins * sizeof(double);

    // ---- generation 0: the live bank; then fission generations until the fission bank is empty ----
    Bank in = A;
    int gen = 0;
    uint64_t n_in = live_total;
    for (;;) {
      st.in_is_birth = gen > 0 ? 1 : 0;
      ta.in = in; ta.census_out = Bk; ta.sec_out = (gen & 1) ? S2 : S1;
      Bank &sec = (gen & 1) ? S2 : S1;
      CK(cudaMemsetAsync(in.cursor, 0, ns * sizeof(uint32_t), p->stream));
      CK(cudaMemsetAsync(sec.count, 0, ns * sizeof(uint32_t), p->stream));
      int grid = (int)std::min<uint64_t>((uint64_t)max_grid, std::max<uint64_t>(1, (n_in + TRANSPORT_THREADS - 1) / TRANSPORT_THREADS));
      CK(cudaEventRecord(ev0, p->stream));
      if (p->last_kernel.compare(0, 11, "k_transport") != 0) p->last_kernel = std::string("k_transport rev=") + MCDC_KERNEL_REV;
      k_transport<<<grid, TRANSPORT_THREADS, smem, p->stream>>>(p->tab, st, ta);
      CK(cudaEventRecord(ev1, p->stream));
      p->launches++;
      CK(cudaMemcpyAsync(h_counts.data(), counts_dev, (size_t)8 * ws_ns * sizeof(uint32_t), cudaMemcpyDeviceToHost, p->stream));
      CK(cudaStreamSynchronize(p->stream));
      CK(cudaGetLastError());
      float ms = 0.f;
      cudaEventElapsedTime(&ms, ev0, ev1);
      p->ms_transport += ms;
      const uint32_t *hc = h_counts.data() + (sec.count - counts_dev);
      uint64_t n_sec = 0;
      for (uint32_t s = 0; s < ns; ++s) {
        if (hc[s] > p->cap) return MCDC_ERR_BANK_OVERFLOW;
        n_sec += hc[s];
      }
      if (n_sec == 0) break;
      in = sec; n_in = n_sec; gen++;
    }
    // census bank becomes the next step's live bank
    {
      const uint32_t *hc = h_counts.data() + (Bk.count - counts_dev);
      live_total = 0;
      for (uint32_t s = 0; s < ns; ++s) {
        if (hc[s] > p->cap) return MCDC_ERR_BANK_OVERFLOW;
        live_total += hc[s];
      }
    }
    if (p->tech.population_control && k < p->K - 1 && live_total > 0) {
      // Appendix G.3: the census bank Bk is controlled into the (consumed) live bank A, batch by batch
      uint32_t n_max = 0;
      {
        const uint32_t *hc = h_counts.data() + (Bk.count - counts_dev);
        for (uint32_t s = 0; s < ns; ++s) n_max = std::max(n_max, hc[s]);
      }
      PcParams pc;
      pc.cap = p->cap; pc.k = k; pc.target = p->tech.pc_target ? p->tech.pc_target : (unsigned long long)sb.hs; pc.w_out = 0.0;
      const dim3 grid((n_max + 255) / 256, ns);
      CK(cudaMemsetAsync(p->d_wfix, 0, ns * sizeof(unsigned long long), p->stream));
      CK(cudaMemsetAsync(A.count, 0, ns * sizeof(uint32_t), p->stream));
      k_pc_weight<<<grid, 256, 0, p->stream>>>(Bk, p->cap, p->d_wfix);
      k_pc_apply<<<grid, 256, 0, p->stream>>>(Bk, A, pc, p->d_wfix, p->d_cnt, p->d_pop_w_after, p->d_pop_n_after);
      p->launches += 2;
      CK(cudaMemcpyAsync(h_counts.data(), counts_dev, (size_t)8 * ws_ns * sizeof(uint32_t), cudaMemcpyDeviceToHost, p->stream));
      CK(cudaStreamSynchronize(p->stream));
      CK(cudaGetLastError());
      const uint32_t *hc = h_counts.data() + (A.count - counts_dev);
      live_total = 0;
      for (uint32_t s = 0; s < ns; ++s) {
        if (hc[s] > p->cap) return MCDC_ERR_BANK_OVERFLOW;
        live_total += hc[s];
      }
    } else {
      std::swap(A, Bk);
    }
    CK(cudaMemsetAsync(Bk.count, 0, ns * sizeof(uint32_t), p->stream));
  }
  if (sb.closeout) {
    int grid = (int)std::min<size_t>((p->n_bins + 255) / 256, (size_t)p->n_sm * 8);
    k_closeout<<<grid, 256, 0, p->stream>>>(p->x_acc, (int)sb.closeout_slots, sb.closeout == 2 ? 1 : 0, p->n_bins, p->d_sum, p->d_sumsq);
    if (p->col_on) { k_closeout<<<grid, 256, 0, p->stream>>>(p->d_xc_acc, (int)sb.closeout_slots, sb.closeout == 2 ? 1 : 0, p->n_bins, p->d_sumc, p->d_sumsqc); p->launches++; }
    p->launches++;
  }
  return MCDC_OK;
}

// ---- k_warp instantiations live in translation units of their own (mcdc_warp_inst.cu, one per VARIANT) ----
enum { KW_ANALOG = 0, KW_WEIGHTED = 1, KW_CENSUS_STEP = 2, KW_GENERATION = 3 };   // VARIANT of k_warp
// SCORE of k_warp for a problem and its merge choice (mcdc_warp.cuh)
// (-1: the instantiation for general CSG regions, Appendix J)
int score_mode(const Tables &T, int aggregate) { return T.has_regions ? -1 : T.all_one_bin ? (aggregate ? 2 : 1) : 0; }
void warp_launch(mcdc_problem *p, bool staged, bool record, int variant, int nt, int grid, size_t smem, cudaStream_t st, const Tables &T, const HistoryArgs &A) {
  const int score = score_mode(T, A.aggregate);
  char name[160];
  snprintf(name, sizeof name, "k_warp<%d,%d,%d,%d,%d%s> rev=%s grid=%d pool_slots=%u smem=%zu", staged ? 1 : 0, record ? 1 : 0, variant,
           score < 0 ? 0 : score, nt, score < 0 ? ",rgn" : "", MCDC_KERNEL_REV, grid, A.pool_slots, smem);
  p->last_kernel = name;
  switch (variant) {
    case KW_ANALOG: warp_launch_variant<KW_ANALOG>(staged, record, score, grid, smem, st, T, A); break;
    case KW_WEIGHTED: warp_launch_variant<KW_WEIGHTED>(staged, record, score, grid, smem, st, T, A); break;
    case KW_CENSUS_STEP: warp_launch_variant<KW_CENSUS_STEP>(staged, record, score, grid, smem, st, T, A); break;
    default: warp_launch_variant<KW_GENERATION>(staged, record, score, grid, smem, st, T, A); break;
  }
}
cudaError_t warp_set_smem(bool staged, bool record, int variant, int score, int nt, int bytes) {
  (void)nt;
  switch (variant) {
    case KW_ANALOG: return warp_set_smem_variant<KW_ANALOG>(staged, record, score, bytes);
    case KW_WEIGHTED: return warp_set_smem_variant<KW_WEIGHTED>(staged, record, score, bytes);
    case KW_CENSUS_STEP: return warp_set_smem_variant<KW_CENSUS_STEP>(staged, record, score, bytes);
    default: return warp_set_smem_variant<KW_GENERATION>(staged, record, score, bytes);
  }
}

// shared-memory plan of k_warp for this problem: stage the hot tables when a pool of at least 64 slots per warp still fits
// in-warp merge of equal tally addresses pays only on tiny meshes (profiles/r01d)
int problem_aggregate(const mcdc_problem *p) { return ((size_t)p->G * p->n_spatial <= 64) ? 1 : 0; }

#ifndef MCDC_POOL_RESERVE
#define MCDC_POOL_RESERVE 8u
#endif
// debug_pool_slots / debug_stage_tables: the documented test knobs of mcdc_run_opts (0 = automatic choice)
int plan_warp_kernel(mcdc_problem *p, bool record, int variant, uint32_t debug_pool_slots = 0, int debug_stage_tables = 0) {
  const bool weighted = variant != KW_ANALOG;
  int dev = 0, max_optin = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
#ifdef MCDC_WARP_SMEM_CAP
  max_optin = std::min(max_optin, MCDC_WARP_SMEM_CAP);
#endif
  const int nt = MCDC_WARP_THREADS;
  const int nw = nt / 32;
  const size_t pop_bytes = align_up((size_t)p->K * 4, 16) + (weighted ? align_up((size_t)p->K * 8 * popw_copies(variant), 16) : 0);
  const size_t fixed = sizeof(WarpShared) + 128 + pop_bytes;
  const size_t hot = align_up(p->tab.hot_bytes, 16);
  const size_t per_slot = warp_pool_bytes_per_slot(record, weighted);
  auto slots = [&](bool staged) -> long {
    const long avail = (long)max_optin - (long)fixed - (long)(staged ? hot : 0);
    if (avail <= 0) return 0;
    long W = avail / (long)(per_slot * nw);
    W = std::min<long>(W, 248L);
    return W / 8 * 8;                                  // keeps every array of the pool 8-byte aligned
  };
  bool staged = slots(true) >= 64;
  if (debug_stage_tables > 0) staged = slots(true) >= 32;
  if (debug_stage_tables < 0) staged = false;
  long W = slots(staged);
  if (debug_pool_slots) W = std::min<long>(W, std::max<long>(32, (long)debug_pool_slots / 8 * 8));
  if (W < 32) return MCDC_ERR_NOMEM;
  p->stage_tables = staged; p->hist_threads = nt; p->pool_slots = (uint32_t)W;
  // slots a refill leaves free for fission children (mcdc_warp.cuh); the debug knob asks for pools that overflow
  // (weighted runs keep particles alive longer -- implicit capture -- and their pools run fuller: with 8 free slots a sixth
  // of the weighted kernel's samples sat in the overflow queue's global loads; 16 took ic_wr from 34.2 to 28.4 ms, while
  // the analog kernel loses 0.6 % with 16)
  p->pool_reserve = debug_pool_slots ? 0u : (weighted ? 2u * MCDC_POOL_RESERVE : MCDC_POOL_RESERVE);
  p->pool_smem = (staged ? hot : 0) + pop_bytes + (size_t)W * nw * per_slot;
  cudaError_t e1 = warp_set_smem(staged, record, variant, score_mode(p->tab, problem_aggregate(p)), nt, (int)p->pool_smem);
  if (e1 != cudaSuccess) return cuda_fail(p, e1, "cudaFuncSetAttribute(k_warp)");
  return MCDC_OK;
}

// the next pair of the handle's launch events (created once, reused by every run)
int next_event_pair(mcdc_problem *p, cudaEvent_t &a, cudaEvent_t &b) {
  if (p->ev_used == p->ev_pairs.size()) {
    cudaEvent_t x = nullptr, y = nullptr;
    CK(cudaEventCreate(&x));
    cudaError_t e = cudaEventCreate(&y);
    if (e != cudaSuccess) { cudaEventDestroy(x); return cuda_fail(p, e, "cudaEventCreate"); }
    p->ev_pairs.emplace_back(x, y);
  }
  a = p->ev_pairs[p->ev_used].first; b = p->ev_pairs[p->ev_used].second;
  p->ev_used++;
  return MCDC_OK;
}
int ensure_run_events(mcdc_problem *p) {
  for (cudaEvent_t *e : {&p->e_run0, &p->e_run1, &p->e_tr0, &p->e_tr1})
    if (!*e) CK(cudaEventCreate(e));
  return MCDC_OK;
}
// sum the device time of the recorded launch pairs (after the stream has been synchronised)
void collect_launch_times(mcdc_problem *p, bool ok) {
  for (size_t i = 0; i < p->ev_used; ++i) {
    float m2 = 0.f;
    if (ok && cudaEventElapsedTime(&m2, p->ev_pairs[i].first, p->ev_pairs[i].second) == cudaSuccess) p->ms_transport += m2;
  }
  p->ev_used = 0;
}

// ---- asynchronous scheduler: one k_warp launch per sub-batch, no host synchronisation ----
int run_subbatch_async(mcdc_problem *p, const SubBatch &sb, uint64_t seed, uint64_t first_history_id, bool record) {
  HistoryArgs ha;
  ha.q = p->queue;
  ha.hist_cursor = p->d_hist_cursor;
  ha.seed_mixed = mix64(seed + MCDC_GAMMA);
  ha.first_history = first_history_id + sb.first_local;
  ha.n_hist = sb.n_hist; ha.hb = sb.hs;
  ha.x_acc = p->x_acc; ha.xc_acc = p->col_on ? p->d_xc_acc : nullptr; ha.cnt = p->d_cnt; ha.pop_w = p->d_pop_w; ha.pop_n = p->d_pop_n;
  ha.ev = record ? p->d_ev + (size_t)sb.first_local * 4 : nullptr;
  ha.aggregate = problem_aggregate(p);   // in-warp merge of equal bins pays only on tiny meshes
  ha.step_mode = 0; ha.step_k = 0; ha.step_source = 1; ha.step_single = 1; ha.bank_cap = 0;
  ha.in = p->bankA; ha.census_out = p->bankB;             // unused outside the census-step mode
  CK(cudaMemsetAsync(p->d_hist_cursor, 0, sizeof(uint32_t), p->stream));
  // consumers' cursor := producers' cursor (drops whatever an aborted launch may have left behind)
  CK(cudaMemcpyAsync(p->d_head_tail, p->d_head_tail + 1, sizeof(unsigned long long), cudaMemcpyDeviceToDevice, p->stream));
  const bool staged = p->stage_tables;
  ha.smem_tables = staged ? (uint32_t)align_up(p->tab.hot_bytes, 16) : 0u;
  ha.pool_slots = p->pool_slots; ha.pool_reserve = p->pool_reserve;
  const size_t smem = p->pool_smem;
  const int nt = p->hist_threads;
  // one block per SM; fewer only when the sub-batch cannot give every warp one full round of 32 histories (small
  // runs are bound by their longest fission chains, so spreading them over all SMs beats filling the pools:
  // 1e5 config-0 histories 0.95 -> 0.68 ms, 1e5 config-3 histories 1.39 -> 1.20 ms)
  const uint64_t per_block = (uint64_t)32 * (nt / 32);
  int grid = (int)std::min<uint64_t>((uint64_t)p->n_sm, std::max<uint64_t>(1, ((uint64_t)sb.n_hist + per_block - 1) / per_block));
  // chunk of source histories a warp reserves at a time: large enough to keep the cursor atomic cold, small enough
  // that the last chunks still spread over all warps
  ha.src_chunk = (uint32_t)std::max<uint64_t>(32, std::min<uint64_t>(128, (uint64_t)sb.n_hist / ((uint64_t)grid * (nt / 32) * 8)));
  ha.n_slots = sb.n_slots;
  ha.n_chunks = sb.n_slots * ((sb.hs + ha.src_chunk - 1) / ha.src_chunk);
  cudaEvent_t a, b;
  { const int rce = next_event_pair(p, a, b); if (rce != MCDC_OK) return rce; }
  CK(cudaEventRecord(a, p->stream));
  const bool weighted = p->tech.implicit_capture || p->tech.wr_threshold > 0.0 || p->col_on;
  warp_launch(p, staged, record, weighted ? KW_WEIGHTED : KW_ANALOG, nt, grid, smem, p->stream, p->tab, ha);
  CK(cudaEventRecord(b, p->stream));
  p->launches++;
  if (sb.closeout) {
    int cgrid = (int)std::min<size_t>((p->n_bins + 255) / 256, (size_t)p->n_sm * 8);
    k_closeout<<<cgrid, 256, 0, p->stream>>>(p->x_acc, (int)sb.closeout_slots, sb.closeout == 2 ? 1 : 0, p->n_bins, p->d_sum, p->d_sumsq);
    if (p->col_on) { k_closeout<<<cgrid, 256, 0, p->stream>>>(p->d_xc_acc, (int)sb.closeout_slots, sb.closeout == 2 ? 1 : 0, p->n_bins, p->d_sumc, p->d_sumsqc); p->launches++; }
    p->launches++;
  }
  CK(cudaGetLastError());
  return MCDC_OK;
}

// ---- population control on the history kernel: one k_warp<WEIGHTED> launch per census step (census-step mode),
// the control kernels between the steps.  Nothing comes back to the host inside the loop: the launches of all census
// steps are queued back to back ("mid-run host <-> device copies" are the cost the paper itself names).
// What the host used to read per step is decided on the device instead: grids are sized for the bank capacity and
// blocks without work leave at once; a bank overflow sets the device flag that mcdc_run_ex checks after the run.
// With K in the thousands that alone would queue thousands of empty launches after the population has died out (or
// after an overflow that is reported only at the end), so past the source every STEP_POLL-th step also copies the next
// step's live counts and the overflow flag to pinned host memory behind an event.  The host looks at a snapshot
// STEP_POLL steps after queueing it, when it has long been made: it never waits for the head of the queue, the launches
// still go out back to back, and at most 2 STEP_POLL steps run on nothing.
constexpr int STEP_POLL = 16;
int run_subbatch_stepwarp(mcdc_problem *p, const SubBatch &sb, uint64_t seed, uint64_t first_history_id, bool record) {
  const uint32_t ns = sb.n_slots, ws_ns = p->ws_slots;
  uint32_t *counts_dev = p->counts_dev;
  CK(cudaMemsetAsync(counts_dev, 0, (size_t)8 * ws_ns * sizeof(uint32_t), p->stream));
  Bank A = p->bankA, Bk = p->bankB;
  const int k_first = step_of(p, p->src_t0), k_last = step_of(p, p->src_t1);
  HistoryArgs ha;
  ha.q = p->queue;
  ha.hist_cursor = p->d_hist_cursor;
  ha.seed_mixed = mix64(seed + MCDC_GAMMA);
  ha.first_history = first_history_id + sb.first_local;
  ha.n_hist = sb.n_hist; ha.hb = sb.hs;
  ha.x_acc = p->x_acc; ha.xc_acc = p->col_on ? p->d_xc_acc : nullptr; ha.cnt = p->d_cnt; ha.pop_w = p->d_pop_w; ha.pop_n = p->d_pop_n;
  ha.ev = record ? p->d_ev + (size_t)sb.first_local * 4 : nullptr;
  ha.aggregate = problem_aggregate(p);
  const bool staged = p->stage_tables;
  ha.smem_tables = staged ? (uint32_t)align_up(p->tab.hot_bytes, 16) : 0u;
  ha.pool_slots = p->pool_slots; ha.pool_reserve = p->pool_reserve;
  const int nt = p->hist_threads;
  const uint64_t per_block = (uint64_t)p->pool_slots * (nt / 32);
  const int grid_src = (int)std::min<uint64_t>((uint64_t)p->n_sm, std::max<uint64_t>(1, ((uint64_t)sb.n_hist + per_block - 1) / per_block));
  ha.src_chunk = (uint32_t)std::max<uint64_t>(32, std::min<uint64_t>(128, (uint64_t)sb.n_hist / ((uint64_t)grid_src * (nt / 32) * 8)));
  ha.n_slots = sb.n_slots;
  ha.step_mode = 1; ha.step_single = (k_first == k_last) ? 1 : 0; ha.bank_cap = p->cap;
  // the population in flight is not known here: as many blocks as the banks could feed (a run of a few thousand
  // histories does not wake every SM), every SM otherwise
  const uint64_t work_max = std::max<uint64_t>((uint64_t)sb.n_hist, (uint64_t)std::min<uint64_t>((uint64_t)p->cap * ns, (uint64_t)4 * sb.n_hist));
  const int grid = (int)std::min<uint64_t>((uint64_t)p->n_sm, std::max<uint64_t>(1, (work_max + per_block - 1) / per_block));
  if (p->h_poll_cap < (size_t)ns + 1) {
    if (p->h_poll) { cudaFreeHost(p->h_poll); p->h_poll = nullptr; p->h_poll_cap = 0; }
    CK(cudaHostAlloc((void **)&p->h_poll, ((size_t)ws_ns + 1) * sizeof(uint32_t), cudaHostAllocDefault));
    p->h_poll_cap = (size_t)ws_ns + 1;
  }
  if (!p->e_poll) CK(cudaEventCreateWithFlags(&p->e_poll, cudaEventDisableTiming));
  bool poll_pending = false;
  for (int k = k_first; k < p->K; ++k) {
    const bool src = k <= k_last;
    ha.step_k = k; ha.step_source = src ? 1 : 0;
    ha.n_chunks = src ? sb.n_slots * ((sb.hs + ha.src_chunk - 1) / ha.src_chunk) : 0u;
    ha.in = A; ha.census_out = Bk;
    CK(cudaMemsetAsync(p->d_hist_cursor, 0, sizeof(uint32_t), p->stream));
    CK(cudaMemcpyAsync(p->d_head_tail, p->d_head_tail + 1, sizeof(unsigned long long), cudaMemcpyDeviceToDevice, p->stream));
    CK(cudaMemsetAsync(A.cursor, 0, ns * sizeof(uint32_t), p->stream));
    cudaEvent_t a, b;
    { const int rce = next_event_pair(p, a, b); if (rce != MCDC_OK) return rce; }
    CK(cudaEventRecord(a, p->stream));
    warp_launch(p, staged, record, KW_CENSUS_STEP, nt, grid, p->pool_smem, p->stream, p->tab, ha);
    CK(cudaEventRecord(b, p->stream));
    p->launches++;
    if (k < p->K - 1) {
      if (p->tech.population_control) {                   // Appendix G.3: census bank Bk -> live bank A
        PcParams pc;
        pc.cap = p->cap; pc.k = k; pc.target = p->tech.pc_target ? p->tech.pc_target : (unsigned long long)sb.hs; pc.w_out = 0.0;
        // (a batch holds at most 4x its source count here unless the caller bound a larger bank: blocks past a
        // slot's count leave at once)
        // in place: the census bank itself becomes the next live bank (survivors keep their records, removed ones are
        // marked as holes, copies are appended behind the arrivals, whose count is frozen in bankS1.count first)
        const dim3 pgrid((p->cap + 255) / 256, ns);
        CK(cudaMemsetAsync(p->d_wfix, 0, ns * sizeof(unsigned long long), p->stream));
        CK(cudaMemcpyAsync(p->bankS1.count, Bk.count, ns * sizeof(uint32_t), cudaMemcpyDeviceToDevice, p->stream));
        k_pc_weight<<<pgrid, 256, 0, p->stream>>>(Bk, p->cap, p->d_wfix);
        k_pc_apply_inplace<<<pgrid, 256, 0, p->stream>>>(Bk, p->bankS1.count, pc, p->d_wfix, p->d_cnt, p->d_pop_w_after, p->d_pop_n_after);
        p->launches += 2;
      }
      std::swap(A, Bk);
    }
    CK(cudaMemsetAsync(Bk.count, 0, ns * sizeof(uint32_t), p->stream));
    if (k > k_last && k < p->K - 1 && (k - k_last) % STEP_POLL == 0) {
      if (poll_pending) {                                  // the snapshot queued STEP_POLL steps ago
        CK(cudaEventSynchronize(p->e_poll));
        bool any_live = false;
        for (uint32_t s = 0; s < ns; ++s) any_live = any_live || p->h_poll[s] != 0u;
        // nothing left to transport and no source to come: every later step would be an empty launch.  Or a bank
        // overflowed: the run is void (mcdc_run_ex reports it), no point in finishing it.  Either way the banks are
        // left as a finished run leaves them (counts zeroed at the next run) and the close-out below still runs.
        if (!any_live || p->h_poll[ns] != 0u) break;
      }
      CK(cudaMemcpyAsync(p->h_poll, A.count, ns * sizeof(uint32_t), cudaMemcpyDeviceToHost, p->stream));   // A: live bank of step k + 1
      CK(cudaMemcpyAsync(p->h_poll + ns, &p->d_cnt->overflow, sizeof(uint32_t), cudaMemcpyDeviceToHost, p->stream));
      CK(cudaEventRecord(p->e_poll, p->stream));
      poll_pending = true;
    }
  }
  if (sb.closeout) {
    int cgrid = (int)std::min<size_t>((p->n_bins + 255) / 256, (size_t)p->n_sm * 8);
    k_closeout<<<cgrid, 256, 0, p->stream>>>(p->x_acc, (int)sb.closeout_slots, sb.closeout == 2 ? 1 : 0, p->n_bins, p->d_sum, p->d_sumsq);
    if (p->col_on) { k_closeout<<<cgrid, 256, 0, p->stream>>>(p->d_xc_acc, (int)sb.closeout_slots, sb.closeout == 2 ? 1 : 0, p->n_bins, p->d_sumc, p->d_sumsqc); p->launches++; }
    p->launches++;
  }
  CK(cudaGetLastError());
  return MCDC_OK;
}

}  // namespace

extern "C" int mcdc_run_ex(mcdc_problem *p, uint64_t n_histories, uint64_t seed, const mcdc_run_opts *opts) {
  if (!p || n_histories == 0) return MCDC_ERR_ARG;
  mcdc_run_opts def = {1u, 0ull, 0, 0, 0u, 0};
  if (!opts) opts = &def;
  const uint32_t B = opts->n_batches ? opts->n_batches : 1u;
  if (n_histories % B != 0) return MCDC_ERR_ARG;
  const uint64_t hb = n_histories / B;
  if (p->batch_size != 0 && p->batch_size != hb) return MCDC_ERR_ARG;
  if (!p->ws) return MCDC_ERR_NO_WORKSPACE;
  if (opts->scheduler != MCDC_SCHED_ASYNC && opts->scheduler != MCDC_SCHED_CENSUS_STEPPED) return MCDC_ERR_ARG;
  // problems outside the compact tables of k_warp (16-bit ids, ...) run on the census-stepped scheduler
  const bool stepped = opts->scheduler == MCDC_SCHED_CENSUS_STEPPED || !p->tab.warp_ok || p->ws_slots > 4095u;
  // the population control needs every particle of a batch parked at the census: the history kernel then runs one
  // launch per census step (census-step mode) with the control kernels in between
  const bool stepwarp = !stepped && p->tech.population_control;
  if ((stepped || stepwarp) && p->cap == 0) return MCDC_ERR_NO_WORKSPACE;   // bound for the asynchronous scheduler only
  const uint64_t slot_max = (stepped || stepwarp) ? std::max<uint64_t>(1, std::min<uint64_t>(p->cap / 2, p->ws_hist)) : p->ws_hist;
  if (p->tech.population_control && hb > slot_max) return MCDC_ERR_ARG;   // the control acts on whole batches
  { const int rcc = ensure_collision_buffers(p); if (rcc != MCDC_OK) return rcc; }
  { const int rce = ensure_run_events(p); if (rce != MCDC_OK) return rce; }
  const bool record = opts->record_history_events != 0;
  if (record) {                                          // the per-history event array is kept and only ever grown
    if (p->ev_cap < n_histories) {
      if (p->d_ev) { cudaFree(p->d_ev); p->d_ev = nullptr; p->ev_cap = 0; }
      CK(cudaMalloc((void **)&p->d_ev, n_histories * 4 * sizeof(uint32_t)));
      p->ev_cap = n_histories;
    }
    CK(cudaMemsetAsync(p->d_ev, 0, n_histories * 4 * sizeof(uint32_t), p->stream));
    p->ev_n = n_histories;
  } else p->ev_n = 0;

  if (stepped) {
    if (!p->transport_attr_set) {
      CK(cudaFuncSetAttribute(k_transport, cudaFuncAttributeMaxDynamicSharedMemorySize, SLAB_MAX_BINS * (int)sizeof(double)));
      p->transport_attr_set = true;
    }
    int occ = 1;   // occupancy with the largest slab this problem can ask for
    size_t per_step = (size_t)p->G * p->n_spatial;
    size_t smem = per_step <= (size_t)SLAB_MAX_BINS ? std::min<size_t>((size_t)SLAB_MAX_BINS, per_step * (size_t)p->Nt) * 8 : 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_transport, TRANSPORT_THREADS, smem) == cudaSuccess && occ > 0)
      p->blocks_per_sm = occ;
  } else {
    const int rcp = plan_warp_kernel(p, record, stepwarp ? KW_CENSUS_STEP
                                     : (p->tech.implicit_capture || p->tech.wr_threshold > 0.0 || p->col_on) ? KW_WEIGHTED : KW_ANALOG,
                                     opts->debug_pool_slots, opts->debug_stage_tables);
    if (rcp != MCDC_OK) return rcp;
  }
  p->ms_transport = 0.0;
  p->ev_used = 0;
  CK(cudaEventRecord(p->e_run0, p->stream));

  // ---- plan sub-batches ----
  auto dispatch = [&](const SubBatch &sb) {
    return stepped ? run_subbatch(p, sb, seed, opts->first_history_id, record)
         : stepwarp ? run_subbatch_stepwarp(p, sb, seed, opts->first_history_id, record)
                    : run_subbatch_async(p, sb, seed, opts->first_history_id, record);
  };
  int rc = MCDC_OK;
  if (hb <= slot_max) {                                  // whole batches, one per slot
    const uint32_t per_sub = (uint32_t)std::max<uint64_t>(1, std::min<uint64_t>(p->ws_slots, p->ws_hist / hb));
    for (uint32_t b = 0; b < B && rc == MCDC_OK; b += per_sub) {
      SubBatch sb;
      sb.n_slots = std::min<uint32_t>(per_sub, B - b);
      sb.first_local = (uint64_t)b * hb; sb.n_hist = (uint32_t)(sb.n_slots * hb); sb.hs = (uint32_t)hb; sb.closeout = 1;
      sb.closeout_slots = sb.n_slots;
      rc = dispatch(sb);
    }
  } else {                                               // one batch = several pieces spread over the slots
    const uint64_t per_sub = std::min<uint64_t>(p->ws_hist, slot_max * p->ws_slots);
    for (uint32_t b = 0; b < B && rc == MCDC_OK; ++b) {
      uint32_t slots_used = 0;                           // most slots any piece of this batch scored into
      for (uint64_t off = 0; off < hb && rc == MCDC_OK; off += per_sub) {
        SubBatch sb;
        uint64_t n = std::min<uint64_t>(per_sub, hb - off);
        sb.hs = (uint32_t)std::min<uint64_t>(slot_max, (n + p->ws_slots - 1) / p->ws_slots);
        sb.n_slots = (uint32_t)((n + sb.hs - 1) / sb.hs);
        sb.first_local = (uint64_t)b * hb + off; sb.n_hist = (uint32_t)n;
        sb.closeout = (off + n >= hb) ? 2 : 0;
        slots_used = std::max(slots_used, sb.n_slots);
        sb.closeout_slots = slots_used;                  // the close-out sums every slot a piece of the batch touched
        rc = dispatch(sb);
      }
    }
  }
  cudaEventRecord(p->e_run1, p->stream);
  cudaError_t se = cudaStreamSynchronize(p->stream);
  float ms = 0.f;
  if (se == cudaSuccess) cudaEventElapsedTime(&ms, p->e_run0, p->e_run1);
  p->ms_run = ms;
  collect_launch_times(p, se == cudaSuccess);
  if (rc != MCDC_OK) return rc;
  if (se != cudaSuccess) return cuda_fail(p, se, "cudaStreamSynchronize");
  int overflow = 0;
  CK(cudaMemcpy(&overflow, &p->d_cnt->overflow, sizeof(int), cudaMemcpyDeviceToHost));
  if (overflow) return MCDC_ERR_BANK_OVERFLOW;
  p->histories += n_histories; p->batches += B; p->batch_size = hb;
  return MCDC_OK;
}

// ---- k-eigenvalue mode (include/mcdc.h mcdc_run_eigenvalue; DESIGN.md Appendix H) ----
extern "C" int mcdc_run_eigenvalue(mcdc_problem *p, uint64_t n_particles, uint64_t seed, uint32_t n_inactive,
                                   uint32_t n_active, double *k_gen) {
  if (!p || !k_gen || n_particles == 0 || n_active == 0 || n_particles > 0x7FFFFFF0ull) return MCDC_ERR_ARG;
  if (p->batch_size != 0 && p->batch_size != n_particles) return MCDC_ERR_ARG;
  if (!p->ws) return MCDC_ERR_NO_WORKSPACE;
  if (!p->tab.warp_ok) return MCDC_ERR_ARG;               // this mode exists on the history kernel only
  if (p->K != 1) return MCDC_ERR_ARG;                     // H.2: one census beyond every flight (a census arrival would be
                                                          // parked in the generation's fission bank)
  if (p->cap == 0 || p->ws_hist < n_particles) return MCDC_ERR_NO_WORKSPACE;
  if (p->tech.population_control) return MCDC_ERR_ARG;    // there is no census here; the generation has its own control
  { const int rcc = ensure_collision_buffers(p); if (rcc != MCDC_OK) return rcc; }
  const int rcp = plan_warp_kernel(p, false, KW_GENERATION);
  if (rcp != MCDC_OK) return rcp;
  const uint32_t ws_ns = p->ws_slots, N = (uint32_t)n_particles;
  uint32_t *counts_dev = p->counts_dev;
  std::vector<uint32_t> h_counts((size_t)8 * ws_ns);
  CK(cudaMemsetAsync(counts_dev, 0, (size_t)8 * ws_ns * sizeof(uint32_t), p->stream));
  Bank A = p->bankA, Bk = p->bankB;
  HistoryArgs ha;
  ha.q = p->queue;
  ha.hist_cursor = p->d_hist_cursor;
  ha.seed_mixed = mix64(seed + MCDC_GAMMA);
  ha.first_history = 0ull;
  ha.n_hist = N; ha.hb = N;
  ha.x_acc = p->x_acc; ha.xc_acc = p->col_on ? p->d_xc_acc : nullptr; ha.cnt = p->d_cnt; ha.pop_w = p->d_pop_w; ha.pop_n = p->d_pop_n;
  ha.ev = nullptr;
  ha.aggregate = problem_aggregate(p);
  const bool staged = p->stage_tables;
  ha.smem_tables = staged ? (uint32_t)align_up(p->tab.hot_bytes, 16) : 0u;
  ha.pool_slots = p->pool_slots; ha.pool_reserve = p->pool_reserve;
  const int nt = p->hist_threads;
  const uint64_t per_block = (uint64_t)p->pool_slots * (nt / 32);
  ha.src_chunk = (uint32_t)std::max<uint64_t>(32, std::min<uint64_t>(128, (uint64_t)N / ((uint64_t)p->n_sm * (nt / 32) * 8)));
  ha.n_slots = 1;
  ha.step_mode = 2; ha.step_k = 0; ha.step_single = 1; ha.bank_cap = p->cap;
  { const int rce = ensure_run_events(p); if (rce != MCDC_OK) return rce; }
  p->ms_transport = 0.0;
  p->ev_used = 0;
  CK(cudaEventRecord(p->e_run0, p->stream));
  const uint32_t G_total = n_inactive + n_active;
  double prod_prev = 0.0, lost_prev = 0.0;
  {
    DevCounters h;
    CK(cudaMemcpy(&h, p->d_cnt, sizeof(h), cudaMemcpyDeviceToHost));
    prod_prev = h.ledger[1]; lost_prev = h.ledger[6];
  }
  uint64_t live = 0;
  int rc = MCDC_OK;
  for (uint32_t g = 0; g < G_total; ++g) {
    ha.step_source = (g == 0) ? 1 : 0;
    ha.n_chunks = (g == 0) ? (N + ha.src_chunk - 1) / ha.src_chunk : 0u;
    ha.in = A; ha.census_out = Bk;
    CK(cudaMemsetAsync(p->d_hist_cursor, 0, sizeof(uint32_t), p->stream));
    CK(cudaMemcpyAsync(p->d_head_tail, p->d_head_tail + 1, sizeof(unsigned long long), cudaMemcpyDeviceToDevice, p->stream));
    CK(cudaMemsetAsync(A.cursor, 0, sizeof(uint32_t), p->stream));
    CK(cudaMemsetAsync(Bk.count, 0, sizeof(uint32_t), p->stream));
    const uint64_t work = (g == 0) ? N : live;
    const int grid = (int)std::min<uint64_t>((uint64_t)p->n_sm, std::max<uint64_t>(1, (work + per_block - 1) / per_block));
    cudaEvent_t a, b;
    { const int rce = next_event_pair(p, a, b); if (rce != MCDC_OK) return rce; }
    CK(cudaEventRecord(a, p->stream));
    warp_launch(p, staged, false, KW_GENERATION, nt, grid, p->pool_smem, p->stream, p->tab, ha);
    CK(cudaEventRecord(b, p->stream));
    p->launches++;
    // H.2: an active generation is one statistical batch; an inactive one is discarded
    if (g >= n_inactive) {
      int cgrid = (int)std::min<size_t>((p->n_bins + 255) / 256, (size_t)p->n_sm * 8);
      k_closeout<<<cgrid, 256, 0, p->stream>>>(p->x_acc, 1, 0, p->n_bins, p->d_sum, p->d_sumsq);
      if (p->col_on) { k_closeout<<<cgrid, 256, 0, p->stream>>>(p->d_xc_acc, 1, 0, p->n_bins, p->d_sumc, p->d_sumsqc); p->launches++; }
      p->launches++;
    } else {
      CK(cudaMemsetAsync(p->x_acc, 0, p->n_bins * sizeof(double), p->stream));
      if (p->col_on) CK(cudaMemsetAsync(p->d_xc_acc, 0, p->n_bins * sizeof(double), p->stream));
    }
    DevCounters h;
    CK(cudaMemcpyAsync(&h, p->d_cnt, sizeof(h), cudaMemcpyDeviceToHost, p->stream));
    CK(cudaMemcpyAsync(h_counts.data(), counts_dev, (size_t)8 * ws_ns * sizeof(uint32_t), cudaMemcpyDeviceToHost, p->stream));
    CK(cudaStreamSynchronize(p->stream));
    CK(cudaGetLastError());
    if (h.overflow) { rc = MCDC_ERR_BANK_OVERFLOW; break; }
    const double start_w = (g == 0) ? (double)N - (h.ledger[6] - lost_prev) : (double)live;   // unit weights (H.3)
    k_gen[g] = start_w > 0.0 ? (h.ledger[1] - prod_prev) / start_w : 0.0;
    prod_prev = h.ledger[1];
    const uint32_t n_fis = h_counts[Bk.count - counts_dev];
    if (n_fis > p->cap) { rc = MCDC_ERR_BANK_OVERFLOW; break; }
    if (g >= n_inactive) { p->histories += N; p->batches += 1; }
    live = 0;
    if (n_fis == 0) { for (uint32_t r = g + 1; r < G_total; ++r) k_gen[r] = 0.0; break; }
    if (g + 1 == G_total) break;
    // H.3: the fission bank Bk is controlled to N particles of weight 1 -> the next generation's bank A
    PcParams pc;
    pc.cap = p->cap; pc.k = 0; pc.target = N; pc.w_out = 1.0;
    const dim3 pgrid((n_fis + 255) / 256, 1);
    CK(cudaMemsetAsync(p->d_wfix, 0, sizeof(unsigned long long), p->stream));
    CK(cudaMemsetAsync(A.count, 0, sizeof(uint32_t), p->stream));
    k_pc_weight<<<pgrid, 256, 0, p->stream>>>(Bk, p->cap, p->d_wfix);
    k_pc_apply<<<pgrid, 256, 0, p->stream>>>(Bk, A, pc, p->d_wfix, p->d_cnt, p->d_pop_w_after, p->d_pop_n_after);
    p->launches += 2;
    CK(cudaMemcpyAsync(h_counts.data(), counts_dev, (size_t)8 * ws_ns * sizeof(uint32_t), cudaMemcpyDeviceToHost, p->stream));
    CK(cudaStreamSynchronize(p->stream));
    CK(cudaGetLastError());
    live = h_counts[A.count - counts_dev];
    if (live > p->cap) { rc = MCDC_ERR_BANK_OVERFLOW; break; }
  }
  cudaEventRecord(p->e_run1, p->stream);
  cudaError_t se = cudaStreamSynchronize(p->stream);
  float ms = 0.f;
  if (se == cudaSuccess) cudaEventElapsedTime(&ms, p->e_run0, p->e_run1);
  p->ms_run = ms;
  collect_launch_times(p, se == cudaSuccess);
  if (se != cudaSuccess) return cuda_fail(p, se, "cudaStreamSynchronize");
  if (rc != MCDC_OK) return rc;
  p->batch_size = n_particles;
  p->ev_n = 0;
  return MCDC_OK;
}

extern "C" int mcdc_run(mcdc_problem *p, uint64_t n_histories, uint64_t seed) {
  return mcdc_run_ex(p, n_histories, seed, nullptr);
}

// =============================================================================================
// results
// =============================================================================================
extern "C" int mcdc_tally_sums_get(const mcdc_problem *cp, double *sum, double *sumsq, size_t n_bins) {
  mcdc_problem *p = const_cast<mcdc_problem *>(cp);
  if (!p || !sum || !sumsq) return MCDC_ERR_ARG;
  if (n_bins != p->n_bins) return MCDC_ERR_SIZE;
  CK(cudaMemcpy(sum, p->d_sum, n_bins * sizeof(double), cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(sumsq, p->d_sumsq, n_bins * sizeof(double), cudaMemcpyDeviceToHost));
  return MCDC_OK;
}

// A.9: mean = sum / N; with m_b = S_b / (N/B): sdev = sqrt((sum m_b^2 / B - mean^2) / (B - 1)); B = 1 -> 0
extern "C" int mcdc_tallies_get(const mcdc_problem *cp, double *mean, double *sdev, size_t n_bins) {
  mcdc_problem *p = const_cast<mcdc_problem *>(cp);
  if (!p || !mean || !sdev) return MCDC_ERR_ARG;
  if (n_bins != p->n_bins) return MCDC_ERR_SIZE;
  if (p->histories == 0) return MCDC_ERR_ARG;
  return batch_statistics(p, p->d_sum, p->d_sumsq, mean, sdev, n_bins);
}

extern "C" int mcdc_counters_get(const mcdc_problem *cp, mcdc_counters *c) {
  mcdc_problem *p = const_cast<mcdc_problem *>(cp);
  if (!p || !c) return MCDC_ERR_ARG;
  DevCounters h;
  CK(cudaMemcpy(&h, p->d_cnt, sizeof(h), cudaMemcpyDeviceToHost));
  c->source = h.ledger[0]; c->production = h.ledger[1]; c->capture = h.ledger[2]; c->fission_abs = h.ledger[3];
  c->leak = h.ledger[4]; c->census_final = h.ledger[5]; c->lost = h.ledger[6];
  c->histories = h.n[0]; c->segments = h.n[1]; c->collisions = h.n[2]; c->surf_hits = h.n[3];
  c->census_events = h.n[4]; c->children = h.n[5]; c->lost_n = h.n[6];
  c->vr_gain = h.ledger[7]; c->vr_loss = h.ledger[8]; c->pc_removed = h.n[7]; c->pc_added = h.n[8];
  c->batches = p->batches; c->kernel_launches = p->launches;
  c->ms_run = p->ms_run; c->ms_transport = p->ms_transport;
  return MCDC_OK;
}

extern "C" int mcdc_census_get(const mcdc_problem *cp, double *pop_w, uint64_t *pop_n, size_t K) {
  mcdc_problem *p = const_cast<mcdc_problem *>(cp);
  if (!p || !pop_w || !pop_n) return MCDC_ERR_ARG;
  if (K != (size_t)p->K) return MCDC_ERR_SIZE;
  CK(cudaMemcpy(pop_w, p->d_pop_w, K * sizeof(double), cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(pop_n, p->d_pop_n, K * sizeof(uint64_t), cudaMemcpyDeviceToHost));
  return MCDC_OK;
}

namespace {
// allocate (or re-allocate after a re-bind with more slots) the collision-estimator accumulators
int ensure_collision_buffers(mcdc_problem *p) {
  if (!p->col_on) return MCDC_OK;
  const uint32_t slots = std::max<uint32_t>(1, p->ws_slots);
  if (p->d_xc_acc && p->xc_slots >= slots) return MCDC_OK;
  if (p->d_xc_acc) { cudaFree(p->d_xc_acc); p->d_xc_acc = nullptr; }
  CK(cudaMalloc((void **)&p->d_xc_acc, (size_t)slots * p->n_bins * sizeof(double)));
  CK(cudaMemset(p->d_xc_acc, 0, (size_t)slots * p->n_bins * sizeof(double)));
  p->xc_slots = slots;
  if (!p->d_sumc) {
    CK(cudaMalloc((void **)&p->d_sumc, p->n_bins * sizeof(double)));
    CK(cudaMalloc((void **)&p->d_sumsqc, p->n_bins * sizeof(double)));
    CK(cudaMemset(p->d_sumc, 0, p->n_bins * sizeof(double)));
    CK(cudaMemset(p->d_sumsqc, 0, p->n_bins * sizeof(double)));
  }
  return MCDC_OK;
}

// A.9 from a pair of device accumulators
int batch_statistics(mcdc_problem *p, const double *d_sum, const double *d_sumsq, double *mean, double *sdev, size_t n_bins) {
  if (n_bins >= (size_t)1 << 18) {                        // large mesh: the per-bin arithmetic runs on the device
    // temporaries: two batch accumulators of the bound workspace when it has them (they are zero between runs and are
    // zeroed again here), else a transient allocation
    double *tmp = nullptr;
    const bool in_ws = p->x_acc && p->ws_slots >= 2;
    if (in_ws) tmp = p->x_acc;
    if (in_ws || cudaMalloc((void **)&tmp, 2 * n_bins * sizeof(double)) == cudaSuccess) {
      const int grid = (int)std::min<size_t>((n_bins + 255) / 256, (size_t)p->n_sm * 16);
      k_statistics<<<grid, 256, 0, p->stream>>>(d_sum, d_sumsq, n_bins, (double)p->histories, (double)p->batches, tmp, tmp + n_bins);
      p->launches++;
      cudaError_t e1 = cudaMemcpyAsync(mean, tmp, n_bins * sizeof(double), cudaMemcpyDeviceToHost, p->stream);
      cudaError_t e2 = cudaMemcpyAsync(sdev, tmp + n_bins, n_bins * sizeof(double), cudaMemcpyDeviceToHost, p->stream);
      if (in_ws) cudaMemsetAsync(tmp, 0, 2 * n_bins * sizeof(double), p->stream);
      cudaError_t e3 = cudaStreamSynchronize(p->stream);
      if (!in_ws) cudaFree(tmp);
      if (e1 != cudaSuccess) return cuda_fail(p, e1, "cudaMemcpyAsync(mean)");
      if (e2 != cudaSuccess) return cuda_fail(p, e2, "cudaMemcpyAsync(sdev)");
      if (e3 != cudaSuccess) return cuda_fail(p, e3, "k_statistics");
      return MCDC_OK;
    }
    cudaGetLastError();                                   // no room for the temporaries: host loop below
  }
  CK(cudaMemcpy(mean, d_sum, n_bins * sizeof(double), cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(sdev, d_sumsq, n_bins * sizeof(double), cudaMemcpyDeviceToHost));
  const double N = (double)p->histories, B = (double)p->batches, hb = N / B;
  for (size_t i = 0; i < n_bins; ++i) {
    double mu = mean[i] / N;
    double sd = 0.0;
    if (B > 1.0) {
      double m2 = sdev[i] / (hb * hb) / B;
      double var = (m2 - mu * mu) / (B - 1.0);
      sd = var > 0.0 ? std::sqrt(var) : 0.0;
    }
    mean[i] = mu; sdev[i] = sd;
  }
  return MCDC_OK;
}
}  // namespace

extern "C" int mcdc_collision_tally_enable(mcdc_problem *p, int on) {
  if (!p) return MCDC_ERR_ARG;
  p->col_on = on ? 1 : 0;
  return MCDC_OK;
}

extern "C" int mcdc_collision_tallies_get(const mcdc_problem *cp, double *mean, double *sdev, size_t n_bins) {
  mcdc_problem *p = const_cast<mcdc_problem *>(cp);
  if (!p || !mean || !sdev) return MCDC_ERR_ARG;
  if (n_bins != p->n_bins) return MCDC_ERR_SIZE;
  if (p->histories == 0 || !p->d_sumc) return MCDC_ERR_ARG;
  return batch_statistics(p, p->d_sumc, p->d_sumsqc, mean, sdev, n_bins);
}

extern "C" int mcdc_census_after_get(const mcdc_problem *cp, double *pop_w, uint64_t *pop_n, size_t K) {
  mcdc_problem *p = const_cast<mcdc_problem *>(cp);
  if (!p || !pop_w || !pop_n) return MCDC_ERR_ARG;
  if (K != (size_t)p->K) return MCDC_ERR_SIZE;
  CK(cudaMemcpy(pop_w, p->d_pop_w_after, K * sizeof(double), cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(pop_n, p->d_pop_n_after, K * sizeof(uint64_t), cudaMemcpyDeviceToHost));
  return MCDC_OK;
}

extern "C" int mcdc_technique_set(mcdc_problem *p, const mcdc_technique *t) {
  if (!p) return MCDC_ERR_ARG;
  mcdc_technique z = {0, 0.0, 0.0, 0, 0ull};
  if (!t) t = &z;
  if (t->wr_threshold > 0.0 && !(t->wr_survive >= t->wr_threshold)) return MCDC_ERR_ARG;
  if (t->wr_threshold < 0.0 || t->wr_threshold != t->wr_threshold) return MCDC_ERR_ARG;
  p->tech = *t;
  p->tab.implicit_capture = t->implicit_capture ? 1 : 0;   // Tables travel by value with every launch
  p->tab.wr_threshold = t->wr_threshold > 0.0 ? t->wr_threshold : 0.0;
  p->tab.wr_survive = t->wr_survive;
  return MCDC_OK;
}

// ---- multi-rank reduction support (include/mcdc.h "Multi-GPU domain replication") ----
namespace {
// sum, sumsq, [sum_c, sumsq_c when the collision-estimator tally is on], pop_w, pop_n, ledger, counts, histories, batches
size_t state_doubles(const mcdc_problem *p) { return (p->col_on ? 4 : 2) * p->n_bins + 2 * (size_t)p->K + 9 + 9 + 2; }
}
extern "C" int mcdc_state_size(const mcdc_problem *p, size_t *n) {
  if (!p || !n) return MCDC_ERR_ARG;
  *n = state_doubles(p);
  return MCDC_OK;
}

extern "C" int mcdc_state_export(const mcdc_problem *cp, double *buf, size_t n, int on_device) {
  mcdc_problem *p = const_cast<mcdc_problem *>(cp);
  if (!p || !buf) return MCDC_ERR_ARG;
  if (n != state_doubles(p)) return MCDC_ERR_SIZE;
  const size_t nb = p->n_bins, K = (size_t)p->K;
  const cudaMemcpyKind big = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  CK(cudaMemcpyAsync(buf, p->d_sum, nb * sizeof(double), big, p->stream));
  CK(cudaMemcpyAsync(buf + nb, p->d_sumsq, nb * sizeof(double), big, p->stream));
  if (p->col_on) {                                        // Appendix I accumulators ride along (allocated on first use)
    { const int rcc = ensure_collision_buffers(p); if (rcc != MCDC_OK) return rcc; }
    CK(cudaMemcpyAsync(buf + 2 * nb, p->d_sumc, nb * sizeof(double), big, p->stream));
    CK(cudaMemcpyAsync(buf + 3 * nb, p->d_sumsqc, nb * sizeof(double), big, p->stream));
    buf += 2 * nb;
  }
  CK(cudaMemcpyAsync(buf + 2 * nb, p->d_pop_w, K * sizeof(double), big, p->stream));
  // the integer tail goes through the host (a few hundred bytes)
  std::vector<unsigned long long> pn(K);
  DevCounters h;
  CK(cudaMemcpyAsync(pn.data(), p->d_pop_n, K * sizeof(unsigned long long), cudaMemcpyDeviceToHost, p->stream));
  CK(cudaMemcpyAsync(&h, p->d_cnt, sizeof(h), cudaMemcpyDeviceToHost, p->stream));
  CK(cudaStreamSynchronize(p->stream));
  std::vector<double> tail(K + 20);
  for (size_t k = 0; k < K; ++k) tail[k] = (double)pn[k];
  for (int e = 0; e < 9; ++e) { tail[K + e] = h.ledger[e]; tail[K + 9 + e] = (double)h.n[e]; }
  tail[K + 18] = (double)p->histories; tail[K + 19] = (double)p->batches;
  double *dst = buf + 2 * nb + K;
  if (on_device) {
    CK(cudaMemcpyAsync(dst, tail.data(), tail.size() * sizeof(double), cudaMemcpyHostToDevice, p->stream));
    CK(cudaStreamSynchronize(p->stream));
  } else std::memcpy(dst, tail.data(), tail.size() * sizeof(double));
  return MCDC_OK;
}

extern "C" int mcdc_state_import(mcdc_problem *p, const double *buf, size_t n, int on_device) {
  if (!p || !buf) return MCDC_ERR_ARG;
  if (n != state_doubles(p)) return MCDC_ERR_SIZE;
  const size_t nb = p->n_bins, K = (size_t)p->K;
  const cudaMemcpyKind big = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  CK(cudaMemcpyAsync(p->d_sum, buf, nb * sizeof(double), big, p->stream));
  CK(cudaMemcpyAsync(p->d_sumsq, buf + nb, nb * sizeof(double), big, p->stream));
  if (p->col_on) {
    { const int rcc = ensure_collision_buffers(p); if (rcc != MCDC_OK) return rcc; }
    CK(cudaMemcpyAsync(p->d_sumc, buf + 2 * nb, nb * sizeof(double), big, p->stream));
    CK(cudaMemcpyAsync(p->d_sumsqc, buf + 3 * nb, nb * sizeof(double), big, p->stream));
    buf += 2 * nb;
  }
  CK(cudaMemcpyAsync(p->d_pop_w, buf + 2 * nb, K * sizeof(double), big, p->stream));
  std::vector<double> tail(K + 20);
  const double *src = buf + 2 * nb + K;
  if (on_device) {
    CK(cudaMemcpyAsync(tail.data(), src, tail.size() * sizeof(double), cudaMemcpyDeviceToHost, p->stream));
    CK(cudaStreamSynchronize(p->stream));
  } else std::memcpy(tail.data(), src, tail.size() * sizeof(double));
  std::vector<unsigned long long> pn(K);
  for (size_t k = 0; k < K; ++k) pn[k] = (unsigned long long)llround(tail[k]);
  DevCounters h;
  std::memset(&h, 0, sizeof(h));
  for (int e = 0; e < 9; ++e) { h.ledger[e] = tail[K + e]; h.n[e] = (unsigned long long)llround(tail[K + 9 + e]); }
  CK(cudaMemcpyAsync(p->d_pop_n, pn.data(), K * sizeof(unsigned long long), cudaMemcpyHostToDevice, p->stream));
  CK(cudaMemcpyAsync(p->d_cnt, &h, sizeof(h), cudaMemcpyHostToDevice, p->stream));
  CK(cudaStreamSynchronize(p->stream));
  p->histories = (uint64_t)llround(tail[K + 18]); p->batches = (uint64_t)llround(tail[K + 19]);
  return MCDC_OK;
}

extern "C" int mcdc_history_events_get(const mcdc_problem *cp, uint32_t *ev, size_t n) {
  mcdc_problem *p = const_cast<mcdc_problem *>(cp);
  if (!p || !ev) return MCDC_ERR_ARG;
  if (n != p->ev_n || !p->d_ev) return MCDC_ERR_SIZE;
  CK(cudaMemcpy(ev, p->d_ev, n * 4 * sizeof(uint32_t), cudaMemcpyDeviceToHost));
  return MCDC_OK;
}

extern "C" int mcdc_problem_info_get(const mcdc_problem *p, mcdc_problem_info *info) {
  if (!p || !info) return MCDC_ERR_ARG;
  info->transmission_halfspaces = p->n_transm; info->certified_halfspaces = p->n_cert;
  info->cells = (uint64_t)p->C; info->one_bin_cells = p->n_one_bin; info->hot_table_bytes = p->tab.hot_bytes;
  info->warp_kernel_ok = p->tab.warp_ok; info->score_fast = p->tab.score_fast;
  info->all_one_bin = p->tab.all_one_bin; info->source_cell = p->tab.src_cell;
  return MCDC_OK;
}

extern "C" const char *mcdc_strerror(int code) {
  switch (code) {
    case MCDC_OK: return "ok";
    case MCDC_ERR_ARG: return "invalid argument";
    case MCDC_ERR_XS: return "inconsistent cross sections";
    case MCDC_ERR_GEOM: return "invalid geometry description";
    case MCDC_ERR_SIZE: return "result buffer size mismatch";
    case MCDC_ERR_NO_WORKSPACE: return "no workspace bound or workspace too small";
    case MCDC_ERR_BANK_OVERFLOW: return "particle bank overflow (bind a larger workspace)";
    case MCDC_ERR_CUDA: return "CUDA error";
    case MCDC_ERR_NOMEM: return "out of host memory";
    case MCDC_ERR_GRID: return "invalid mesh, time or census grid";
    default: return "unknown error";
  }
}

extern "C" const char *mcdc_last_cuda_error(const mcdc_problem *p) { return p ? p->cuda_err.c_str() : ""; }

extern "C" const char *mcdc_version(void) { return "0.2 sm_100a"; }

extern "C" int mcdc_kernel_info_get(const mcdc_problem *p, char *buf, size_t n) {
  if (!p || !buf || n == 0) return MCDC_ERR_ARG;
  // + how many fission children have gone through the global ring queue since the handle was created (the producers'
  // cursor is monotonic over launches): the evidence that a run took the overflow path
  unsigned long long tail = 0ull;
  if (p->d_head_tail && !p->last_kernel.empty() && p->last_kernel[2] == 'w')
    cudaMemcpy(&tail, p->d_head_tail + 1, sizeof tail, cudaMemcpyDeviceToHost);
  if (p->last_kernel.empty()) snprintf(buf, n, "%s", "");
  else snprintf(buf, n, "%s queue_children=%llu", p->last_kernel.c_str(), tail);
  return MCDC_OK;
}

// ---------------------------------------------------------------------------------------------
// mcdc_tallies_get_noalloc (include/mcdc.h): the A.9 read-out of k_statistics for callers that must not
// allocate device memory.  The 2 * n_bins doubles that batch_statistics() takes from the workspace or from
// cudaMalloc live here in a fixed array of the library's device image instead.
//
// g_noalloc_scratch is that array.  In HOST code the name is only a handle for the runtime, not a device
// address: handing `g_noalloc_scratch` itself to a kernel would make the kernel fault (or, on a GPU that can
// reach host memory, scribble on whatever host address the stand-in happens to have).  Host code therefore
// asks the runtime for the device address once per GPU (noalloc_scratch_address) and passes THAT to the kernel.
// ---------------------------------------------------------------------------------------------
#include <mutex>

static __device__ __align__(256) double g_noalloc_scratch[2 * MCDC_NOALLOC_MAX_BINS];   // [0, MAX) mean, [MAX, 2 MAX) sdev

namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
double *g_noalloc_addr[NOALLOC_MAX_DEVICES];   // device address of g_noalloc_scratch on GPU d; nullptr = not looked up yet
std::mutex g_noalloc_mu;

// Device address of the scratch array on GPU `dev`, which must be the calling thread's current device (every GPU
// has its own copy of the array at its own address).  The first call per GPU asks the runtime; later calls read the cache.
cudaError_t noalloc_scratch_address(int dev, double **out) {
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_addr[dev]) {
    double *ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (!ptr) return cudaErrorInvalidSymbol;
    g_noalloc_addr[dev] = ptr;
  }
  *out = g_noalloc_addr[dev];
  return cudaSuccess;
}
}  // namespace

extern "C" int mcdc_tallies_get_noalloc(const mcdc_problem *cp, double *mean, double *sdev, size_t n_bins) {
  mcdc_problem *p = const_cast<mcdc_problem *>(cp);
  if (!p || !mean || !sdev) return MCDC_ERR_ARG;
  if (n_bins != p->n_bins) return MCDC_ERR_SIZE;
  if (n_bins > MCDC_NOALLOC_MAX_BINS) {
    p->cuda_err = "mcdc_tallies_get_noalloc: the problem has " + std::to_string(n_bins) + " tally bins, the fixed scratch "
                  "array holds MCDC_NOALLOC_MAX_BINS = " + std::to_string((size_t)MCDC_NOALLOC_MAX_BINS) +
                  "; use mcdc_tallies_get with a two-slot workspace for this mesh";
    return MCDC_ERR_SIZE;
  }
  if (p->histories == 0) return MCDC_ERR_ARG;
  // the handle's accumulators live on the GPU that was current at mcdc_problem_create; the scratch address we need is
  // that GPU's, and the look-up below answers for the CURRENT one -- so the two must be the same
  int dev = -1;
  CK(cudaGetDevice(&dev));
  cudaPointerAttributes attr;
  CK(cudaPointerGetAttributes(&attr, p->d_sum));
  if (attr.device != dev || dev < 0 || dev >= NOALLOC_MAX_DEVICES) {
    p->cuda_err = "mcdc_tallies_get_noalloc: the handle lives on GPU " + std::to_string(attr.device) +
                  " but the current device is " + std::to_string(dev);
    return MCDC_ERR_ARG;
  }
  double *scratch = nullptr;
  cudaError_t es = noalloc_scratch_address(dev, &scratch);
  if (es != cudaSuccess) return cuda_fail(p, es, "cudaGetSymbolAddress(g_noalloc_scratch)");
  double *d_mean = scratch, *d_sdev = scratch + MCDC_NOALLOC_MAX_BINS;
  // k_statistics writes mean[i] and sdev[i] for every i < n_bins before anything reads them: what an earlier call
  // left in the array is overwritten, nothing needs clearing.  Same launch shape as batch_statistics().
  const int grid = (int)std::min<size_t>((n_bins + 255) / 256, (size_t)p->n_sm * 16);
  k_statistics<<<grid, 256, 0, p->stream>>>(p->d_sum, p->d_sumsq, n_bins, (double)p->histories, (double)p->batches, d_mean, d_sdev);
  cudaError_t e0 = cudaGetLastError();
  p->launches++;
  cudaError_t e1 = cudaMemcpyAsync(mean, d_mean, n_bins * sizeof(double), cudaMemcpyDeviceToHost, p->stream);
  cudaError_t e2 = cudaMemcpyAsync(sdev, d_sdev, n_bins * sizeof(double), cudaMemcpyDeviceToHost, p->stream);
  cudaError_t e3 = cudaStreamSynchronize(p->stream);
  if (e0 != cudaSuccess) return cuda_fail(p, e0, "k_statistics launch");
  if (e1 != cudaSuccess) return cuda_fail(p, e1, "cudaMemcpyAsync(mean)");
  if (e2 != cudaSuccess) return cuda_fail(p, e2, "cudaMemcpyAsync(sdev)");
  if (e3 != cudaSuccess) return cuda_fail(p, e3, "k_statistics");
  return MCDC_OK;
}
