// mcdc_device.cuh -- device functions of the transport engine (sm_100a).
// RNG, geometry (A.3-A.5), collision physics (A.6).
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include "mcdc_types.h"

namespace mcdc {

#define MCDC_FULL 0xFFFFFFFFu

// ------------------------------------------------------------------------------------------------
// RNG: counter-based, keyed by a 64-bit particle key; draw index = particle counter (Appendix B).
// ------------------------------------------------------------------------------------------------
__host__ __device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
  z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
  z ^= z >> 27; z *= 0x94D049BB133111EBull;
  z ^= z >> 31;
  return z;
}
#define MCDC_GAMMA 0x9E3779B97F4A7C15ull

__device__ __forceinline__ unsigned long long child_key(unsigned long long kp, uint32_t c0, uint32_t j) {
  return mix64(kp + MCDC_GAMMA * ((((unsigned long long)c0) << 8) | (unsigned long long)(j + 1u)));
}

// Philox4x32-10 on counter (block, 0, 0, 0); returns the two 64-bit halves (o1:o0) and (o3:o2).
__device__ __forceinline__ void philox_block(unsigned long long key, uint32_t block,
                                             unsigned long long &lo64, unsigned long long &hi64) {
  uint32_t c0 = block, c1 = 0u, c2 = 0u, c3 = 0u;
  uint32_t k0 = (uint32_t)key, k1 = (uint32_t)(key >> 32);
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  lo64 = ((unsigned long long)c1 << 32) | c0;
  hi64 = ((unsigned long long)c3 << 32) | c2;
}

// u = ((x >> 12) + 0.5) * 2^-52, built exactly: [1,2) mantissa trick then one exact subtraction.
__device__ __forceinline__ double u64_to_unit(unsigned long long x) {
  double d = __longlong_as_double((long long)((x >> 12) | 0x3FF0000000000000ull));
  return d - 0.99999999999999988897769753748434595763683319091796875;   // 1 - 2^-53
}

__device__ __forceinline__ double draw(unsigned long long key, uint32_t &ctr) {
  unsigned long long lo, hi;
  philox_block(key, ctr >> 1, lo, hi);
  unsigned long long x = (ctr & 1u) ? hi : lo;
  ctr += 1u;
  return u64_to_unit(x);
}
// two consecutive draws; when ctr is even they come from one Philox block
__device__ __forceinline__ void draw2(unsigned long long key, uint32_t &ctr, double &a, double &b) {
  unsigned long long lo, hi;
  philox_block(key, ctr >> 1, lo, hi);
  if (ctr & 1u) {
    a = u64_to_unit(hi);
    philox_block(key, (ctr + 1u) >> 1, lo, hi);
    b = u64_to_unit(lo);
  } else {
    a = u64_to_unit(lo); b = u64_to_unit(hi);
  }
  ctr += 2u;
}

// isotropic direction (A.3): mu = 2 xi - 1, phi = 2 pi xi
__device__ __forceinline__ void isotropic(double xi_mu, double xi_phi, double &ux, double &uy, double &uz) {
  double mu = 2.0 * xi_mu - 1.0;
  double st = sqrt(1.0 - mu * mu);
  double s, c;
  sincospi(2.0 * xi_phi, &s, &c);
  ux = st * c; uy = st * s; uz = mu;
}

// first index with xi < cdf[i]; fallback `last`
__device__ __forceinline__ int sample_cdf(const double *__restrict__ cdf, int n, int last, double xi) {
  for (int i = 0; i < n; ++i)
    if (xi < __ldg(cdf + i)) return i;
  return last;
}

// ------------------------------------------------------------------------------------------------
// Geometry
// ------------------------------------------------------------------------------------------------
struct Vec3 { double x, y, z; };

__device__ __forceinline__ double4 ldg_d4(const double4 *p) {
  const double2 a = __ldg((const double2 *)p), b = __ldg((const double2 *)p + 1);
  return make_double4(a.x, a.y, b.x, b.y);
}

__device__ __forceinline__ double quad_f(const double *__restrict__ c, double x, double y, double z) {
  return __ldg(c + 0) * x * x + __ldg(c + 1) * y * y + __ldg(c + 2) * z * z + __ldg(c + 3) * x * y +
         __ldg(c + 4) * x * z + __ldg(c + 5) * y * z + __ldg(c + 6) * x + __ldg(c + 7) * y + __ldg(c + 8) * z +
         __ldg(c + 9);
}
__device__ __forceinline__ Vec3 quad_grad(const double *__restrict__ c, double x, double y, double z) {
  Vec3 g;
  g.x = 2.0 * __ldg(c + 0) * x + __ldg(c + 3) * y + __ldg(c + 4) * z + __ldg(c + 6);
  g.y = 2.0 * __ldg(c + 1) * y + __ldg(c + 3) * x + __ldg(c + 5) * z + __ldg(c + 7);
  g.z = 2.0 * __ldg(c + 2) * z + __ldg(c + 4) * x + __ldg(c + 5) * y + __ldg(c + 8);
  return g;
}

// smallest positive root of a u^2 + 2 k u + c (half-b form) per A.4: q = -(k + sign(k) sqrt(k^2 - a c)), roots q/a and c/q
__device__ __forceinline__ double quad_root(double a, double k, double c) {
  const double INF = CUDART_INF;
  if (a == 0.0) {
    if (k == 0.0) return INF;
    double u = -c / (2.0 * k);
    return (u > 0.0) ? u : INF;
  }
  double disc = k * k - a * c;
  if (disc < 0.0) return INF;
  const double sq = sqrt(disc);
  const double q = (k < 0.0) ? (sq - k) : -(k + sq);      // sign(+-0) = +1 as in A.4
  double best = INF;
  double u1 = q / a;
  if (u1 > 0.0) best = u1;
  if (q != 0.0) {
    double u2 = c / q;
    if (u2 > 0.0 && u2 < best) best = u2;
  }
  return best;
}

// same roots for a > 0 (cylinders): only the root that is the smallest positive one is divided out.
//   c > 0: both roots share the sign of -k; the smaller is c/q.   c < 0: one positive root, q/a if k < 0 else c/q.
//   c == 0 (on the surface): roots 0 and -2k/a.
__device__ __forceinline__ double quad_root_pos_a(double a, double k, double c) {
  const double INF = CUDART_INF;
  if (!(a > 0.0)) return INF;                              // parallel to the axis (A.4 plane branch with b = 0)
  const double disc = k * k - a * c;
  if (disc < 0.0) return INF;
  const double sq = sqrt(disc);
  const double q = (k < 0.0) ? (sq - k) : -(k + sq);      // -(k + sign(k) sqrt(disc)), sign(+-0) = +1 as in A.4
  double u;
  if (c > 0.0) {
    if (k >= 0.0) return INF;
    u = c / q;
  } else if (c < 0.0) {
    u = (k < 0.0) ? q / a : c / q;
  } else {
    if (k >= 0.0) return INF;
    u = q / a;
  }
  return (u > 0.0) ? u : INF;
}

// distance to surface s along (ux,uy,uz) from (x,y,z); on => the particle sits on s (c := 0)
__device__ __forceinline__ double surf_distance(const Tables &T, int s, int type, bool on, double x, double y, double z,
                                                double ux, double uy, double uz, double ix, double iy, double iz) {
  // (ix, iy, iz) = 1 / (ux, uy, uz), computed once per segment
  const double INF = CUDART_INF;
  if (type <= ST_PLANE_Z) {
    if (on) return INF;
    const double pos = __ldg((const double *)(T.surf_q + s));
    double r = (type == ST_PLANE_X) ? x : ((type == ST_PLANE_Y) ? y : z);
    double iu = (type == ST_PLANE_X) ? ix : ((type == ST_PLANE_Y) ? iy : iz);
    double d = (pos - r) * iu;                     // u == 0: iu = inf -> +-inf or NaN, both rejected below
    return (d > 0.0 && d < INF) ? d : INF;
  }
  const double4 q = ldg_d4(T.surf_q + s);
  if (type == ST_CYL_Z) {
    double dx = x - q.x, dy = y - q.y;
    double a = ux * ux + uy * uy;
    double k = dx * ux + dy * uy;
    double c = on ? 0.0 : (dx * dx + dy * dy - q.z);
    return quad_root_pos_a(a, k, c);
  }
  const double *c = T.surf_coef + 10 * s;
  double a = __ldg(c + 0) * ux * ux + __ldg(c + 1) * uy * uy + __ldg(c + 2) * uz * uz + __ldg(c + 3) * ux * uy +
             __ldg(c + 4) * ux * uz + __ldg(c + 5) * uy * uz;
  Vec3 g = quad_grad(c, x, y, z);
  double b = g.x * ux + g.y * uy + g.z * uz;
  double cc = on ? 0.0 : quad_f(c, x, y, z);
  return quad_root(a, 0.5 * b, cc);
}

// sense (+1 / -1) of surface s at r for a particle travelling along u (A.3 tie rule); from_dir forces
// the direction rule (the surface just crossed, A.5)
__device__ __forceinline__ int surf_sense(const Tables &T, int s, int type, bool from_dir, double x, double y, double z,
                                          double ux, double uy, double uz) {
  const double4 q = ldg_d4(T.surf_q + s);
  double f, b;
  if (type <= ST_PLANE_Z) {
    double r = (type == ST_PLANE_X) ? x : ((type == ST_PLANE_Y) ? y : z);
    double u = (type == ST_PLANE_X) ? ux : ((type == ST_PLANE_Y) ? uy : uz);
    f = q.y * (r - q.x); b = q.y * u;
  } else if (type == ST_CYL_Z) {
    double dx = x - q.x, dy = y - q.y;
    f = q.w * (dx * dx + dy * dy - q.z); b = q.w * (dx * ux + dy * uy);
  } else {
    const double *c = T.surf_coef + 10 * s;
    f = quad_f(c, x, y, z);
    Vec3 g = quad_grad(c, x, y, z);
    b = g.x * ux + g.y * uy + g.z * uz;
  }
  if (!from_dir) {
    if (f > 0.0) return 1;
    if (f < 0.0) return -1;
  }
  return (b < 0.0) ? -1 : 1;
}

__device__ __forceinline__ bool cell_contains(const Tables &T, int c, int crossed, double x, double y, double z,
                                              double ux, double uy, double uz) {
  const int e = __ldg(T.cell_off + c + 1);
  for (int i = __ldg(T.cell_off + c); i < e; ++i) {
    int h = __ldg(T.hs + i);                            // packed: surface << 4 | type << 1 | (sense > 0)
    int s = h >> 4, want = (h & 1) ? 1 : -1;
    if (surf_sense(T, s, (h >> 1) & 7, s == crossed, x, y, z, ux, uy, uz) != want) return false;
  }
  return true;
}

// full search in increasing cell id (A.3); slow path
__device__ __noinline__ int locate_all(const Tables &T, int crossed, double x, double y, double z, double ux,
                                       double uy, double uz) {
  for (int c = 0; c < T.C; ++c)
    if (cell_contains(T, c, crossed, x, y, z, ux, uy, uz)) return c;
  return -1;
}

// cell after crossing the surface of half-space slot `slot` of the current cell (A.5, transmission)
__device__ __forceinline__ int locate_neighbour(const Tables &T, int slot, int s_star, double x, double y, double z,
                                                double ux, double uy, double uz) {
  const int e = __ldg(T.nb_off + slot + 1);
  for (int i = __ldg(T.nb_off + slot); i < e; ++i) {
    int c = __ldg(T.nb_cell + i);
    if (cell_contains(T, c, s_star, x, y, z, ux, uy, uz)) return c;
  }
  return locate_all(T, s_star, x, y, z, ux, uy, uz);
}

// source-particle location through the locator grid over the source box
__device__ __forceinline__ int locate_source(const Tables &T, double x, double y, double z, double ux, double uy,
                                             double uz) {
  int v[3];
  const double r[3] = {x, y, z};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    int i = (int)floor((r[a] - T.loc_lo[a]) * T.loc_inv_d[a]);
    v[a] = min(max(i, 0), T.loc_n[a] - 1);
  }
  int vox = (v[2] * T.loc_n[1] + v[1]) * T.loc_n[0] + v[0];
  const int e = __ldg(T.loc_off + vox + 1);
  for (int i = __ldg(T.loc_off + vox); i < e; ++i) {
    int c = __ldg(T.loc_cell + i);
    if (cell_contains(T, c, -1, x, y, z, ux, uy, uz)) return c;
  }
  return locate_all(T, -1, x, y, z, ux, uy, uz);
}

// specular reflection about grad f at the hit point (A.5)
__device__ __forceinline__ void reflect(const Tables &T, int s, int type, double x, double y, double z, double &ux,
                                        double &uy, double &uz) {
  if (type == ST_PLANE_X) { ux = -ux; return; }
  if (type == ST_PLANE_Y) { uy = -uy; return; }
  if (type == ST_PLANE_Z) { uz = -uz; return; }
  Vec3 g = quad_grad(T.surf_coef + 10 * s, x, y, z);
  double inv = 1.0 / sqrt(g.x * g.x + g.y * g.y + g.z * g.z);
  double nx = g.x * inv, ny = g.y * inv, nz = g.z * inv;
  double dot = ux * nx + uy * ny + uz * nz;
  ux -= 2.0 * dot * nx; uy -= 2.0 * dot * ny; uz -= 2.0 * dot * nz;
}

}  // namespace mcdc
