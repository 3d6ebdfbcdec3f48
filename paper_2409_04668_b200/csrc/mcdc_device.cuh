// mcdc_device.cuh -- device functions of the transport engine (sm_100a).
// RNG, table access, geometry (A.3-A.5).
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include "mcdc_types.h"

namespace mcdc {

#define MCDC_FULL 0xFFFFFFFFu

// dynamic shared memory of the transport kernels (staged tables first, kernel-specific data after)
extern __shared__ __align__(16) unsigned char g_smem[];

// ------------------------------------------------------------------------------------------------
// Table accessor.  STAGED = true: the blob's hot prefix was copied to the start of dynamic shared memory
// and every table read is an LDS; false: reads go to the global blob (L1/L2 cached).
// ------------------------------------------------------------------------------------------------
template <bool STAGED>
struct TB {
  const Tables &T;
  __device__ __forceinline__ explicit TB(const Tables &t) : T(t) {}
  template <class V>
  __device__ __forceinline__ V ld(uint32_t off, int i) const {
    if (STAGED) return reinterpret_cast<const V *>(g_smem + off)[i];
    return reinterpret_cast<const V *>(T.blob + off)[i];
  }
  // load at an absolute byte offset of the blob
  template <class V>
  __device__ __forceinline__ V ldb(uint32_t byte_off) const {
    if (STAGED) return *reinterpret_cast<const V *>(g_smem + byte_off);
    return *reinterpret_cast<const V *>(T.blob + byte_off);
  }
  __device__ __forceinline__ double sig_t(int mg) const { return ld<double>(T.o_sig_t, mg); }
  __device__ __forceinline__ double inv_sig_t(int mg) const { return ld<double>(T.o_inv_sig_t, mg); }
  __device__ __forceinline__ double sig_s_tot(int mg) const { return ld<double>(T.o_sig_s_tot, mg); }
  __device__ __forceinline__ double sig_sc(int mg) const { return ld<double>(T.o_sig_sc, mg); }
  __device__ __forceinline__ double sig_f(int mg) const { return ld<double>(T.o_sig_f, mg); }
  __device__ __forceinline__ double nu(int mg) const { return ld<double>(T.o_nu, mg); }
  __device__ __forceinline__ double cap_frac(int mg) const { return ld<double>(T.o_cap_frac, mg); }
  __device__ __forceinline__ double cdf_s(int i) const { return ld<double>(T.o_cdf_s, i); }
  __device__ __forceinline__ int last_s(int mg) const { return ld<int>(T.o_last_s, mg); }
  __device__ __forceinline__ double cdf_chi(int i) const { return ld<double>(T.o_cdf_chi, i); }
  __device__ __forceinline__ int last_chi(int m) const { return ld<int>(T.o_last_chi, m); }
  __device__ __forceinline__ double speed(int g) const { return ld<double>(T.o_speed, g); }
  __device__ __forceinline__ double inv_speed(int g) const { return ld<double>(T.o_inv_speed, g); }
  __device__ __forceinline__ double time_edge(int i) const { return ld<double>(T.o_T, i); }
  __device__ __forceinline__ double census(int k) const { return ld<double>(T.o_census, k); }
  __device__ __forceinline__ double src_cdf(int g) const { return ld<double>(T.o_src_cdf, g); }
  __device__ __forceinline__ double2 surf_q01(int s) const { return ld<double2>(T.o_surf_q, 2 * s); }
  __device__ __forceinline__ double2 surf_q23(int s) const { return ld<double2>(T.o_surf_q, 2 * s + 1); }
  __device__ __forceinline__ double surf_q0(int s) const { return ld<double>(T.o_surf_q, 4 * s); }
  __device__ __forceinline__ int surf_bc(int s) const { return ld<int>(T.o_surf_bc, s); }
  __device__ __forceinline__ int cell_off(int c) const { return ld<int>(T.o_cell_off, c); }
  __device__ __forceinline__ int hs(int i) const { return ld<int>(T.o_hs, i); }
  __device__ __forceinline__ int cell_mat(int c) const { return ld<int>(T.o_cell_mat, c); }
  __device__ __forceinline__ int nb_off(int i) const { return ld<int>(T.o_nb_off, i); }
  __device__ __forceinline__ int nb_cell(int i) const { return ld<int>(T.o_nb_cell, i); }
  __device__ __forceinline__ int loc_off(int i) const { return ld<int>(T.o_loc_off, i); }
  __device__ __forceinline__ int loc_cell(int i) const { return ld<int>(T.o_loc_cell, i); }
  // general quadric coefficients: from shared memory only when they are part of the staged prefix
  __device__ __forceinline__ double coef(int s, int j) const {
    if (STAGED && T.o_surf_coef < T.hot_bytes) return reinterpret_cast<const double *>(g_smem + T.o_surf_coef)[10 * s + j];
    return reinterpret_cast<const double *>(T.blob + T.o_surf_coef)[10 * s + j];
  }
};

__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// fp64 add to a tally accumulator in global memory as a true reduction (REDG): atomicAdd() with an unused result compiles
// to ATOMG with a discarded destination, which still waits for its reply before the same thread can issue the next one --
// the DDA scorer of config 2 spent 37 % of its samples there, one L2 / DRAM round trip per tally bin (profiles/r02n)
__device__ __forceinline__ void red_add_f64(double *p, double v) { asm volatile("red.global.add.f64 [%0], %1;" ::"l"(p), "d"(v)); }

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
// Not inlined: ~80 instructions called from a handful of sites keeps the kernels inside the i-cache.
static __device__ __noinline__ ulonglong2 philox_block(unsigned long long key, uint32_t block) {
  uint32_t c0 = block, c1 = 0u, c2 = 0u, c3 = 0u;
  uint32_t k0 = (uint32_t)key, k1 = (uint32_t)(key >> 32);
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    // high and low word of each product: the compiler pairs them into one IMAD.WIDE.U32 (written as a 64-bit product
    // it added a zero to every high word: 21 more instructions per block, 4 % of the history kernel's instructions)
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  ulonglong2 r;
  r.x = ((unsigned long long)c1 << 32) | c0;
  r.y = ((unsigned long long)c3 << 32) | c2;
  return r;
}

// u = ((x >> 12) + 0.5) * 2^-52, built exactly: [1,2) mantissa trick then one exact subtraction.
__device__ __forceinline__ double u64_to_unit(unsigned long long x) {
  double d = __longlong_as_double((long long)((x >> 12) | 0x3FF0000000000000ull));
  return d - 0.99999999999999988897769753748434595763683319091796875;   // 1 - 2^-53
}

__device__ __forceinline__ double draw(unsigned long long key, uint32_t &ctr) {
  const ulonglong2 b = philox_block(key, ctr >> 1);
  const unsigned long long x = (ctr & 1u) ? b.y : b.x;
  ctr += 1u;
  return u64_to_unit(x);
}
// two consecutive draws; when ctr is even they come from one Philox block
__device__ __forceinline__ void draw2(unsigned long long key, uint32_t &ctr, double &a, double &b) {
  ulonglong2 blk = philox_block(key, ctr >> 1);
  if (ctr & 1u) {
    a = u64_to_unit(blk.y);
    blk = philox_block(key, (ctr + 1u) >> 1);
    b = u64_to_unit(blk.x);
  } else {
    a = u64_to_unit(blk.x); b = u64_to_unit(blk.y);
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

// ------------------------------------------------------------------------------------------------
// Geometry
// ------------------------------------------------------------------------------------------------
struct Vec3 { double x, y, z; };

template <class TBT>
__device__ __forceinline__ double quad_f(const TBT &tb, int s, double x, double y, double z) {
  return tb.coef(s, 0) * x * x + tb.coef(s, 1) * y * y + tb.coef(s, 2) * z * z + tb.coef(s, 3) * x * y +
         tb.coef(s, 4) * x * z + tb.coef(s, 5) * y * z + tb.coef(s, 6) * x + tb.coef(s, 7) * y + tb.coef(s, 8) * z +
         tb.coef(s, 9);
}
template <class TBT>
__device__ __forceinline__ Vec3 quad_grad(const TBT &tb, int s, double x, double y, double z) {
  Vec3 g;
  g.x = 2.0 * tb.coef(s, 0) * x + tb.coef(s, 3) * y + tb.coef(s, 4) * z + tb.coef(s, 6);
  g.y = 2.0 * tb.coef(s, 1) * y + tb.coef(s, 3) * x + tb.coef(s, 5) * z + tb.coef(s, 7);
  g.z = 2.0 * tb.coef(s, 2) * z + tb.coef(s, 4) * x + tb.coef(s, 5) * y + tb.coef(s, 8);
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
  const double disc = k * k - a * c;
  // no root ahead: parallel to the axis (A.4 plane branch with b = 0), no real root, or both roots behind (c >= 0, k >= 0)
  if (!(a > 0.0) || disc < 0.0 || (c >= 0.0 && k >= 0.0)) return INF;
  const double sq = sqrt(disc);
  const double q = (k < 0.0) ? (sq - k) : -(k + sq);      // -(k + sign(k) sqrt(disc)), sign(+-0) = +1 as in A.4
  const bool c_over_q = (c > 0.0) || (c < 0.0 && !(k < 0.0));
  const double u = (c_over_q ? c : q) / (c_over_q ? q : a);   // one division for whichever root is the one ahead
  return (u > 0.0) ? u : INF;
}

// distance to surface s along (ux,uy,uz) from (x,y,z); on => the particle sits on s (c := 0);
// (ix, iy, iz) = 1 / (ux, uy, uz), computed once per segment
template <class TBT>
__device__ __forceinline__ double surf_distance(const TBT &tb, int s, int type, bool on, double x, double y, double z,
                                                double ux, double uy, double uz, double ix, double iy, double iz) {
  const double INF = CUDART_INF;
  if (type <= ST_PLANE_Z) {
    if (on) return INF;
    const double pos = tb.surf_q0(s);
    double r = (type == ST_PLANE_X) ? x : ((type == ST_PLANE_Y) ? y : z);
    double iu = (type == ST_PLANE_X) ? ix : ((type == ST_PLANE_Y) ? iy : iz);
    double d = (pos - r) * iu;                     // u == 0: iu = inf -> +-inf or NaN, both rejected below
    return (d > 0.0 && d < INF) ? d : INF;
  }
  if (type == ST_CYL_Z) {
    const double2 q01 = tb.surf_q01(s);
    const double r2 = tb.surf_q23(s).x;
    double dx = x - q01.x, dy = y - q01.y;
    double a = ux * ux + uy * uy;
    double k = dx * ux + dy * uy;
    double c = on ? 0.0 : (dx * dx + dy * dy - r2);
    return quad_root_pos_a(a, k, c);
  }
  double a = tb.coef(s, 0) * ux * ux + tb.coef(s, 1) * uy * uy + tb.coef(s, 2) * uz * uz + tb.coef(s, 3) * ux * uy +
             tb.coef(s, 4) * ux * uz + tb.coef(s, 5) * uy * uz;
  Vec3 g = quad_grad(tb, s, x, y, z);
  double b = g.x * ux + g.y * uy + g.z * uz;
  double cc = on ? 0.0 : quad_f(tb, s, x, y, z);
  return quad_root(a, 0.5 * b, cc);
}

// sense (+1 / -1) of surface s at r for a particle travelling along u (A.3 tie rule); from_dir forces
// the direction rule (the surface just crossed, A.5)
template <class TBT>
__device__ __forceinline__ int surf_sense(const TBT &tb, int s, int type, bool from_dir, double x, double y, double z,
                                          double ux, double uy, double uz) {
  double f, b;
  if (type <= ST_PLANE_Z) {
    const double2 q = tb.surf_q01(s);
    double r = (type == ST_PLANE_X) ? x : ((type == ST_PLANE_Y) ? y : z);
    double u = (type == ST_PLANE_X) ? ux : ((type == ST_PLANE_Y) ? uy : uz);
    f = q.y * (r - q.x); b = q.y * u;
  } else if (type == ST_CYL_Z) {
    const double2 q01 = tb.surf_q01(s), q23 = tb.surf_q23(s);
    double dx = x - q01.x, dy = y - q01.y;
    f = q23.y * (dx * dx + dy * dy - q23.x); b = q23.y * (dx * ux + dy * uy);
  } else {
    f = quad_f(tb, s, x, y, z);
    Vec3 g = quad_grad(tb, s, x, y, z);
    b = g.x * ux + g.y * uy + g.z * uz;
  }
  if (!from_dir) {
    if (f > 0.0) return 1;
    if (f < 0.0) return -1;
  }
  return (b < 0.0) ? -1 : 1;
}

// RGN: the problem may hold general CSG regions (Appendix J).  The history kernel never runs such problems, and its
// slow paths are instantiated with RGN = false: code it never executes would still cost it instruction-cache room
// (adding the expression evaluator to them slowed the analog kernel by 5 %, profiles/r01f).
template <bool RGN, class TBT>
__device__ __forceinline__ bool cell_contains(const TBT &tb, int c, int crossed, double x, double y, double z,
                                              double ux, double uy, double uz) {
  const int e = tb.cell_off(c + 1);
  if (RGN && tb.T.has_regions) {                               // Appendix J: the cell may be a postfix expression
    const int *off = reinterpret_cast<const int *>(tb.T.blob + tb.T.o_rgn_off);
    const int *tok = reinterpret_cast<const int *>(tb.T.blob + tb.T.o_rgn_tok);
    const int k1 = off[c + 1];
    int k = off[c];
    if (k < k1) {
      const int base = tb.cell_off(c);
      uint32_t st = 0u;                                 // bit stack, top = bit 0 (depth <= 32 checked at create)
      for (; k < k1; ++k) {
        const int t = tok[k];
        if (t >= 0) {
          const int h = tb.hs(base + t);
          const int s = h >> 6, want = (h & 1) ? 1 : -1;
          st = (st << 1) | (surf_sense(tb, s, (h >> 1) & 7, s == crossed, x, y, z, ux, uy, uz) == want ? 1u : 0u);
        } else if (t == -3) st ^= 1u;
        else {
          const uint32_t b = st & 1u;
          st >>= 1;
          st = (t == -1) ? (st & (0xFFFFFFFEu | b)) : (st | b);
        }
      }
      return (st & 1u) != 0u;
    }
  }
  for (int i = tb.cell_off(c); i < e; ++i) {
    const int h = tb.hs(i);                             // packed: surface << 6 | bc << 4 | type << 1 | (sense > 0)
    const int s = h >> 6, want = (h & 1) ? 1 : -1;
    if (surf_sense(tb, s, (h >> 1) & 7, s == crossed, x, y, z, ux, uy, uz) != want) return false;
  }
  return true;
}

// full search in increasing cell id (A.3); slow path.  Not inlined, and it works on the device-memory copy of
// the tables so that no caller has to take the address of its kernel parameter block.
template <bool RGN>
static __device__ __noinline__ int locate_all_dev(const Tables *gT, int crossed, double x, double y, double z, double ux,
                                           double uy, double uz) {
  const TB<false> tb(*gT);
  for (int c = 0; c < gT->C; ++c)
    if (cell_contains<RGN>(tb, c, crossed, x, y, z, ux, uy, uz)) return c;
  return -1;
}
template <bool RGN, class TBT>
__device__ __forceinline__ int locate_all(const TBT &tb, int crossed, double x, double y, double z, double ux, double uy,
                                          double uz) {
  return locate_all_dev<RGN>(tb.T.self_dev, crossed, x, y, z, ux, uy, uz);
}

// cell after crossing the surface of half-space slot `slot` of the current cell (A.5, transmission)
template <bool RGN, class TBT>
__device__ __forceinline__ int locate_neighbour(const TBT &tb, int slot, int s_star, double x, double y, double z,
                                                double ux, double uy, double uz) {
  const int e = tb.nb_off(slot + 1);
  for (int i = tb.nb_off(slot); i < e; ++i) {
    const int c = tb.nb_cell(i);
    if (cell_contains<RGN>(tb, c, s_star, x, y, z, ux, uy, uz)) return c;
  }
  return locate_all<RGN>(tb, s_star, x, y, z, ux, uy, uz);
}

// source-particle location through the locator grid over the source box
template <bool RGN, class TBT>
__device__ __forceinline__ int locate_source(const TBT &tb, double x, double y, double z, double ux, double uy,
                                             double uz) {
  const Tables &T = tb.T;
  int v[3];
  const double r[3] = {x, y, z};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    int i = (int)floor((r[a] - T.loc_lo[a]) * T.loc_inv_d[a]);
    v[a] = min(max(i, 0), T.loc_n[a] - 1);
  }
  const int vox = (v[2] * T.loc_n[1] + v[1]) * T.loc_n[0] + v[0];
  const int e = tb.loc_off(vox + 1);
  for (int i = tb.loc_off(vox); i < e; ++i) {
    const int c = tb.loc_cell(i);
    if (cell_contains<RGN>(tb, c, -1, x, y, z, ux, uy, uz)) return c;
  }
  return locate_all<RGN>(tb, -1, x, y, z, ux, uy, uz);
}

// specular reflection about grad f at the hit point (A.5)
template <class TBT>
__device__ __forceinline__ void reflect(const TBT &tb, int s, int type, double x, double y, double z, double &ux,
                                        double &uy, double &uz) {
  if (type == ST_PLANE_X) { ux = -ux; return; }
  if (type == ST_PLANE_Y) { uy = -uy; return; }
  if (type == ST_PLANE_Z) { uz = -uz; return; }
  Vec3 g = quad_grad(tb, s, x, y, z);
  double inv = 1.0 / sqrt(g.x * g.x + g.y * g.y + g.z * g.z);
  double nx = g.x * inv, ny = g.y * inv, nz = g.z * inv;
  double dot = ux * nx + uy * ny + uz * nz;
  ux -= 2.0 * dot * nx; uy -= 2.0 * dot * ny; uz -= 2.0 * dot * nz;
}

}  // namespace mcdc
