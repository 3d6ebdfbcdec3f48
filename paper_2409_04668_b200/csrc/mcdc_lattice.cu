// mcdc_lattice.cu -- universes and lattices (include/mcdc.h; DESIGN.md Appendix K): host code that expands an nx x ny
// lattice of universes into the flat surfaces / cells of mcdc_problem_desc and hands them to mcdc_problem_create.
// No kernels here: a lattice is an input convenience, the history kernel sees ordinary cells (and proves its
// certified neighbours on them as for any other geometry).
#include <cstdint>
#include <new>
#include <vector>

#include "../../include/mcdc.h"

namespace {

struct Flat {
  std::vector<double> coef;                 // [S][10]
  std::vector<int32_t> bc, cell_off, hs_s, hs_n, mat;
};

bool lattice_ok(const mcdc_lattice_desc *L) {
  if (!L || L->n_universes < 1 || L->nx < 1 || L->ny < 1) return false;
  if (!L->usurf_offset || !L->ucell_offset || !L->uhs_offset || !L->ucell_material || !L->fill) return false;
  if (!(L->pitch_x > 0.0) || !(L->pitch_y > 0.0) || !(L->z_hi > L->z_lo)) return false;
  const int U = L->n_universes;
  if (L->usurf_offset[0] != 0 || L->ucell_offset[0] != 0 || L->uhs_offset[0] != 0) return false;
  for (int u = 0; u < U; ++u) {
    if (L->usurf_offset[u + 1] < L->usurf_offset[u] || L->ucell_offset[u + 1] <= L->ucell_offset[u]) return false;
    const int ns = L->usurf_offset[u + 1] - L->usurf_offset[u];
    for (int c = L->ucell_offset[u]; c < L->ucell_offset[u + 1]; ++c) {
      if (L->uhs_offset[c + 1] <= L->uhs_offset[c]) return false;           // an empty cell
      if (!L->uhs_surface || !L->uhs_sense) return false;
      for (int h = L->uhs_offset[c]; h < L->uhs_offset[c + 1]; ++h) {
        const int s = L->uhs_surface[h];
        if (s >= ns || s < MCDC_LAT_ZHI) return false;
        if (L->uhs_sense[h] != 1 && L->uhs_sense[h] != -1) return false;
      }
    }
  }
  if (L->usurf_offset[U] > 0 && !L->usurf_coef) return false;
  const long long n_elem = (long long)L->nx * L->ny;                         // nx * ny overflows int from 46341 x 46341
  if (n_elem > INT32_MAX) return false;
  for (long long k = 0; k < n_elem; ++k)
    if (L->fill[k] < 0 || L->fill[k] >= U) return false;
  for (int f = 0; f < 6; ++f)
    if (L->bc[f] < MCDC_BC_TRANSMISSION || L->bc[f] > MCDC_BC_REFLECTIVE) return false;
  return true;
}

// Sizes of the flat geometry, in 64 bits; false when any of them does not fit the int32 fields of mcdc_problem_desc.
// Shared by all three entry points, so that none of them expands a lattice whose sizes it could not state.
bool flat_sizes(const mcdc_lattice_desc *L, long long &S, long long &C, long long &H) {
  S = (long long)L->nx + 1 + (long long)L->ny + 1 + 2; C = 0; H = 0;
  const long long n_elem = (long long)L->nx * L->ny;
  for (long long k = 0; k < n_elem; ++k) {
    const int u = L->fill[k];
    S += L->usurf_offset[u + 1] - L->usurf_offset[u];
    C += L->ucell_offset[u + 1] - L->ucell_offset[u];
    H += L->uhs_offset[L->ucell_offset[u + 1]] - L->uhs_offset[L->ucell_offset[u]];
  }
  return S <= INT32_MAX && C <= INT32_MAX && H <= INT32_MAX;
}

void put_plane(Flat &F, int axis, double a, int bc) {
  const size_t o = F.coef.size();
  F.coef.resize(o + 10, 0.0);
  F.coef[o + 6 + axis] = 1.0;
  F.coef[o + 9] = -a;
  F.bc.push_back(bc);
}

// Appendix K.2: f(r - c) for f = A x^2 + B y^2 + C z^2 + D xy + E xz + F yz + G x + H y + I z + J
void put_translated(Flat &F, const double *q, double cx, double cy, double cz) {
  const double A = q[0], B = q[1], C = q[2], D = q[3], E = q[4], Fq = q[5], G = q[6], H = q[7], I = q[8], J = q[9];
  const size_t o = F.coef.size();
  F.coef.resize(o + 10, 0.0);
  double *t = &F.coef[o];
  t[0] = A; t[1] = B; t[2] = C; t[3] = D; t[4] = E; t[5] = Fq;
  t[6] = G - 2.0 * A * cx - D * cy - E * cz;
  t[7] = H - 2.0 * B * cy - D * cx - Fq * cz;
  t[8] = I - 2.0 * C * cz - E * cx - Fq * cy;
  const double quad = A * cx * cx + B * cy * cy + C * cz * cz + D * cx * cy + E * cx * cz + Fq * cy * cz;
  const double lin = G * cx + H * cy + I * cz;
  t[9] = J + quad - lin;
  F.bc.push_back(MCDC_BC_TRANSMISSION);
}

// Appendix K.1 / K.3
void expand(const mcdc_lattice_desc *L, Flat &F) {
  const int nx = L->nx, ny = L->ny;
  for (int i = 0; i <= nx; ++i) put_plane(F, 0, L->x0 + i * L->pitch_x, i == 0 ? L->bc[0] : i == nx ? L->bc[1] : MCDC_BC_TRANSMISSION);
  for (int j = 0; j <= ny; ++j) put_plane(F, 1, L->y0 + j * L->pitch_y, j == 0 ? L->bc[2] : j == ny ? L->bc[3] : MCDC_BC_TRANSMISSION);
  const int oy = nx + 1, oz = nx + 1 + ny + 1;
  put_plane(F, 2, L->z_lo, L->bc[4]);
  put_plane(F, 2, L->z_hi, L->bc[5]);
  std::vector<int32_t> first((size_t)nx * ny);
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      const int u = L->fill[(size_t)j * nx + i];
      first[(size_t)j * nx + i] = (int32_t)F.bc.size();
      const double cx = L->x0 + (i + 0.5) * L->pitch_x, cy = L->y0 + (j + 0.5) * L->pitch_y;
      for (int s = L->usurf_offset[u]; s < L->usurf_offset[u + 1]; ++s) put_translated(F, L->usurf_coef + (size_t)10 * s, cx, cy, 0.0);
    }
  F.cell_off.push_back(0);
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      const int u = L->fill[(size_t)j * nx + i];
      const int32_t face[6] = {i, i + 1, oy + j, oy + j + 1, oz, oz + 1};
      for (int c = L->ucell_offset[u]; c < L->ucell_offset[u + 1]; ++c) {
        for (int h = L->uhs_offset[c]; h < L->uhs_offset[c + 1]; ++h) {
          const int s = L->uhs_surface[h];
          F.hs_s.push_back(s >= 0 ? first[(size_t)j * nx + i] + s : face[-1 - s]);
          F.hs_n.push_back(L->uhs_sense[h]);
        }
        F.cell_off.push_back((int32_t)F.hs_s.size());
        F.mat.push_back(L->ucell_material[c]);
      }
    }
}

}  // namespace

extern "C" int mcdc_lattice_expand_size(const mcdc_lattice_desc *lat, int32_t *n_surfaces, int32_t *n_cells, int32_t *n_halfspaces) {
  if (!n_surfaces || !n_cells || !n_halfspaces) return MCDC_ERR_ARG;
  if (!lattice_ok(lat)) return MCDC_ERR_GEOM;
  long long S, C, H;
  if (!flat_sizes(lat, S, C, H)) return MCDC_ERR_GEOM;
  *n_surfaces = (int32_t)S; *n_cells = (int32_t)C; *n_halfspaces = (int32_t)H;
  return MCDC_OK;
}

extern "C" int mcdc_lattice_expand(const mcdc_lattice_desc *lat, double *surf_coef, int32_t *surf_bc, int32_t *cell_offset,
                                   int32_t *hs_surface, int32_t *hs_sense, int32_t *cell_material) {
  if (!surf_coef || !surf_bc || !cell_offset || !hs_surface || !hs_sense || !cell_material) return MCDC_ERR_ARG;
  if (!lattice_ok(lat)) return MCDC_ERR_GEOM;
  long long S, C, H;
  if (!flat_sizes(lat, S, C, H)) return MCDC_ERR_GEOM;
  Flat F;
  try { expand(lat, F); } catch (const std::bad_alloc &) { return MCDC_ERR_NOMEM; }
  std::copy(F.coef.begin(), F.coef.end(), surf_coef);
  std::copy(F.bc.begin(), F.bc.end(), surf_bc);
  std::copy(F.cell_off.begin(), F.cell_off.end(), cell_offset);
  std::copy(F.hs_s.begin(), F.hs_s.end(), hs_surface);
  std::copy(F.hs_n.begin(), F.hs_n.end(), hs_sense);
  std::copy(F.mat.begin(), F.mat.end(), cell_material);
  return MCDC_OK;
}

extern "C" int mcdc_problem_create_lattice(const mcdc_problem_desc *d, const mcdc_lattice_desc *lat, mcdc_problem **out) {
  if (!d || !out) return MCDC_ERR_ARG;
  if (!lattice_ok(lat)) return MCDC_ERR_GEOM;
  long long S, C, H;
  if (!flat_sizes(lat, S, C, H)) return MCDC_ERR_GEOM;
  Flat F;
  try { expand(lat, F); } catch (const std::bad_alloc &) { return MCDC_ERR_NOMEM; }
  mcdc_problem_desc e = *d;                              // materials, source, mesh, time grid: the caller's
  e.n_surfaces = (int32_t)F.bc.size(); e.n_cells = (int32_t)F.mat.size();
  e.surf_coef = F.coef.data(); e.surf_bc = F.bc.data();
  e.cell_offset = F.cell_off.data(); e.hs_surface = F.hs_s.data(); e.hs_sense = F.hs_n.data();
  e.cell_material = F.mat.data();
  return mcdc_problem_create(&e, out);                   // deep-copies: F may go
}
