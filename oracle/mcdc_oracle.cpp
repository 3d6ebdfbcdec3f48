// mcdc_oracle.cpp -- ORACLE: test infrastructure, not product.  parity pinned (tests/test_oracle_*.py).
//
// Plain single-threaded fp64 restatement of the time-dependent multigroup Monte Carlo history
// loop, step by step in the order and notation of SURVEY.md
// Appendix A (transport) and Appendix B (RNG).  No blocking, fusion or reordering; build with
// -O2 -ffp-contract=off.  Shares nothing with the CUDA path.
#include "mcdc_oracle.h"

#include <cmath>
#include <cstdint>
#include <cstring>
#include <deque>
#include <limits>
#include <vector>

namespace {

const double INF = std::numeric_limits<double>::infinity();
const double PI = 3.14159265358979323846;

// ---------------------------------------------------------------------------------------------
// Appendix B: RNG.  gamma, the 64-bit finaliser M, Philox4x32-10 (Salmon et al., SC'11).
// ---------------------------------------------------------------------------------------------
const uint64_t GAMMA = 0x9E3779B97F4A7C15ull;

uint64_t mix64(uint64_t z) {
  z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
  z ^= z >> 27; z *= 0x94D049BB133111EBull;
  z ^= z >> 31;
  return z;
}

void philox4x32_10(const uint32_t c_in[4], const uint32_t k_in[2], uint32_t out[4]) {
  uint32_t c0 = c_in[0], c1 = c_in[1], c2 = c_in[2], c3 = c_in[3];
  uint32_t k0 = k_in[0], k1 = k_in[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;   // multiplier on word 0
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;   // multiplier on word 2
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;       // key schedule (bumped after every round)
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

uint64_t source_key(uint64_t seed, uint64_t h) { return mix64(mix64(seed + GAMMA) ^ h); }

uint64_t child_key(uint64_t kp, uint32_t c0, uint32_t j) {
  return mix64(kp + GAMMA * ((((uint64_t)c0) << 8) | (uint64_t)(j + 1)));
}

// draw(p): block = ctr>>1; x64 = (ctr&1) ? (o3:o2) : (o1:o0); u = ((x64>>12)+0.5)*2^-52; ctr++
double draw(uint64_t key, uint32_t &ctr) {
  uint32_t c[4] = {ctr >> 1, 0u, 0u, 0u};
  uint32_t k[2] = {(uint32_t)(key & 0xFFFFFFFFull), (uint32_t)(key >> 32)};
  uint32_t o[4];
  philox4x32_10(c, k, o);
  uint64_t x64 = (ctr & 1u) ? (((uint64_t)o[3] << 32) | o[2]) : (((uint64_t)o[1] << 32) | o[0]);
  ctr += 1;
  return ((double)(x64 >> 12) + 0.5) * (1.0 / 4503599627370496.0);   // 2^-52
}

// ---------------------------------------------------------------------------------------------
// A.1 data
// ---------------------------------------------------------------------------------------------
struct Surface { double A, B, C, D, E, F, G, H, I, J; int bc; };

struct Particle {
  double x, y, z, ux, uy, uz, t, w;
  int g, cell, last_surface;
  uint64_t key; uint32_t ctr;
  int k;                       // index (0-based) of the next census time
  bool alive;
};

struct BankItem {              // a source particle or a fission birth record (A.6)
  bool is_birth;
  Particle p;                  // for a birth record only x,y,z,t,w,cell,key,k are meaningful
};

}  // namespace

struct orc_problem {
  int G, M, S, C;
  std::vector<double> sigma_t, sigma_c, sigma_f, nu, chi, sigma_s, sigma_s_tot, speed;
  std::vector<Surface> surf;
  std::vector<int> cell_offset, hs_surface, hs_sense, cell_material;
  std::vector<double> bb_lo, bb_hi;          // per-cell culling boxes [C][3] (A.5 allows culling)
  // Appendix J: general CSG regions.  Cell c with rgn_off[c] < rgn_off[c+1] is the postfix expression
  // rgn_tok[rgn_off[c] .. rgn_off[c+1]) over its half-spaces (token t >= 0: half-space t of the cell's list holds;
  // -1 AND, -2 OR, -3 NOT); an empty range (or no region table) is the plain intersection of A.1.
  std::vector<int> rgn_off, rgn_tok;
  double src_lo[3], src_hi[3], src_t0, src_t1;
  std::vector<double> src_pdf;
  int src_dir_mode; double src_dir[3];
  double mesh_lo[3], mesh_hi[3]; int mesh_n[3];
  int Nt; std::vector<double> T;
  int K;  std::vector<double> census;
  size_t n_bins;
  // results
  std::vector<double> x, sum, sumsq;         // batch accumulator, sum of S_b, sum of S_b^2
  int col_on;                                // collision-estimator tally (Appendix I) on the same mesh
  std::vector<double> xc, sumc, sumsqc;
  std::vector<double> pop_w; std::vector<uint64_t> pop_n;
  std::vector<double> pop_w_after; std::vector<uint64_t> pop_n_after;   // after the population control (G.3)
  orc_technique tech;                        // Appendix G of DESIGN.md; all zero = analog
  orc_counters cnt;
  uint64_t batch_size;                       // histories per batch (must agree over runs)
  std::vector<uint32_t> hist_ev;             // [n][4] of the last run
  uint32_t *cur_ev;                          // event counters of the history in flight (or null)
};

namespace {

// f(r), grad f(r) for the general quadric (A.1)
inline double f_eval(const Surface &s, double x, double y, double z) {
  return s.A * x * x + s.B * y * y + s.C * z * z + s.D * x * y + s.E * x * z + s.F * y * z +
         s.G * x + s.H * y + s.I * z + s.J;
}
inline void grad_eval(const Surface &s, double x, double y, double z, double g[3]) {
  g[0] = 2.0 * s.A * x + s.D * y + s.E * z + s.G;
  g[1] = 2.0 * s.B * y + s.D * x + s.F * z + s.H;
  g[2] = 2.0 * s.C * z + s.E * x + s.F * y + s.I;
}

// A.4: distance along omega from r to surface s; on_surface => c := 0
double surface_distance(const Surface &s, const double r[3], const double o[3], bool on_surface) {
  double a = s.A * o[0] * o[0] + s.B * o[1] * o[1] + s.C * o[2] * o[2] + s.D * o[0] * o[1] +
             s.E * o[0] * o[2] + s.F * o[1] * o[2];
  double g[3]; grad_eval(s, r[0], r[1], r[2], g);
  double b = g[0] * o[0] + g[1] * o[1] + g[2] * o[2];
  double c = on_surface ? 0.0 : f_eval(s, r[0], r[1], r[2]);
  if (a == 0.0) {                                  // plane
    if (b == 0.0) return INF;
    double u = -c / b;
    return (u > 0.0) ? u : INF;
  }
  double disc = b * b - 4.0 * a * c;
  if (disc < 0.0) return INF;
  double sgn = (b < 0.0) ? -1.0 : 1.0;             // sign(0) = +1
  double q = -0.5 * (b + sgn * std::sqrt(disc));
  double best = INF;
  double u1 = q / a;
  if (u1 > 0.0 && u1 < best) best = u1;
  if (q != 0.0) {
    double u2 = c / q;
    if (u2 > 0.0 && u2 < best) best = u2;
  }
  return best;
}

// sense of surface s at r for a particle travelling along o (A.3): sign f, tie -> sign(grad f . o)
int sense_at(const Surface &s, const double r[3], const double o[3], bool force_direction) {
  double v = force_direction ? 0.0 : f_eval(s, r[0], r[1], r[2]);
  if (v > 0.0) return +1;
  if (v < 0.0) return -1;
  double g[3]; grad_eval(s, r[0], r[1], r[2], g);
  double b = g[0] * o[0] + g[1] * o[1] + g[2] * o[2];
  return (b < 0.0) ? -1 : +1;
}

// A.3 / A.5 locate: first cell (increasing id) all of whose half-spaces hold.  crossed >= 0:
// the sense of that surface is taken from the direction of travel, never from sign f.
int locate(const orc_problem &P, const double r[3], const double o[3], int crossed) {
  for (int c = 0; c < P.C; ++c) {
    bool out = false;                              // culling box (loose: never rejects a true hit)
    for (int a = 0; a < 3; ++a)
      if (r[a] < P.bb_lo[3 * c + a] || r[a] > P.bb_hi[3 * c + a]) { out = true; break; }
    if (out) continue;
    bool ok = true;
    if (!P.rgn_off.empty() && P.rgn_off[c] < P.rgn_off[c + 1]) {      // Appendix J: evaluate the postfix expression
      std::vector<char> st;
      const int base = P.cell_offset[c];
      for (int k = P.rgn_off[c]; k < P.rgn_off[c + 1]; ++k) {
        int t = P.rgn_tok[k];
        if (t >= 0) {
          int s = P.hs_surface[base + t];
          st.push_back(sense_at(P.surf[s], r, o, s == crossed) == P.hs_sense[base + t]);
        } else if (t == -3) { st.back() = !st.back(); }
        else { char b = st.back(); st.pop_back(); st.back() = (t == -1) ? (st.back() && b) : (st.back() || b); }
      }
      ok = st.back() != 0;
    } else {
      for (int i = P.cell_offset[c]; i < P.cell_offset[c + 1]; ++i) {
        int s = P.hs_surface[i];
        if (sense_at(P.surf[s], r, o, s == crossed) != P.hs_sense[i]) { ok = false; break; }
      }
    }
    if (ok) return c;
  }
  return -1;
}

// isotropic direction from two draws (A.3): mu = 2 xi - 1, phi = 2 pi xi
inline void isotropic(double xi_mu, double xi_phi, double &ux, double &uy, double &uz) {
  double mu = 2.0 * xi_mu - 1.0;
  double phi = 2.0 * PI * xi_phi;
  double st = std::sqrt(1.0 - mu * mu);
  ux = st * std::cos(phi); uy = st * std::sin(phi); uz = mu;
}

// first index with xi < running cumulative sum; fallback: last index with a non-zero entry
inline int sample_cdf(const double *pdf, int n, double xi_scaled) {
  double run = 0.0; int last = 0;
  for (int i = 0; i < n; ++i) {
    run += pdf[i];
    if (pdf[i] != 0.0) last = i;
    if (xi_scaled < run) return i;
  }
  return last;
}

inline int first_census_after(const orc_problem &P, double t) {   // smallest k with C[k] > t (D15: else K-1)
  for (int k = 0; k < P.K; ++k) if (P.census[k] > t) return k;
  return P.K - 1;
}

// ---------------------------------------------------------------------------------------------
// A.7 track-length scoring: 4-D DDA over (x, y, z, t) from the pre-move state.
// bin(it, g, iz, iy, ix) += w * length of the piece inside that bin.
// ---------------------------------------------------------------------------------------------
void score_track(orc_problem &P, const Particle &p, double d) {
  const double r[3] = {p.x, p.y, p.z}, o[3] = {p.ux, p.uy, p.uz};
  const double v = P.speed[p.g];
  double u_in = 0.0, u_out = d;
  for (int a = 0; a < 3; ++a) {                       // clip to the mesh box
    double lo = P.mesh_lo[a], hi = P.mesh_hi[a];
    if (o[a] == 0.0) {
      if (!(lo <= r[a] && r[a] < hi)) return;
    } else {
      double u0 = (lo - r[a]) / o[a], u1 = (hi - r[a]) / o[a];
      if (o[a] < 0.0) { double tmp = u0; u0 = u1; u1 = tmp; }
      if (u0 > u_in) u_in = u0;
      if (u1 < u_out) u_out = u1;
    }
  }
  {                                                   // clip to [T[0], T[Nt]]; time at u is t + u/v
    double u0 = (P.T[0] - p.t) * v, u1 = (P.T[P.Nt] - p.t) * v;
    if (u0 > u_in) u_in = u0;
    if (u1 < u_out) u_out = u1;
  }
  if (!(u_in < u_out)) return;

  int idx[3]; double delta[3];
  for (int a = 0; a < 3; ++a) {
    int n = P.mesh_n[a];
    if (n == 1) { idx[a] = 0; delta[a] = P.mesh_hi[a] - P.mesh_lo[a]; continue; }
    delta[a] = (P.mesh_hi[a] - P.mesh_lo[a]) / (double)n;
    double q = std::floor((r[a] + u_in * o[a] - P.mesh_lo[a]) / delta[a]);
    int i = (q < 0.0) ? 0 : ((q > (double)(n - 1)) ? n - 1 : (int)q);
    idx[a] = i;
  }
  int it;                                             // largest it with T[it] <= t + u_in / v
  {
    double t_in = p.t + u_in / v;
    it = 0;
    for (int j = 0; j < P.Nt; ++j) if (P.T[j] <= t_in) it = j;
  }

  double u_cur = u_in;
  for (;;) {
    double cross[4];
    for (int a = 0; a < 3; ++a) {
      if (o[a] == 0.0) { cross[a] = INF; continue; }
      if (P.mesh_n[a] == 1) {                         // single (possibly unbounded) bin: edge = box face
        double edge = (o[a] > 0.0) ? P.mesh_hi[a] : P.mesh_lo[a];
        cross[a] = (edge - r[a]) / o[a];
        continue;
      }
      double edge = (o[a] > 0.0) ? P.mesh_lo[a] + (double)(idx[a] + 1) * delta[a]
                                 : P.mesh_lo[a] + (double)idx[a] * delta[a];
      cross[a] = (edge - r[a]) / o[a];
    }
    cross[3] = (P.T[it + 1] - p.t) * v;
    double u_next = u_out;
    for (int a = 0; a < 4; ++a) if (cross[a] < u_next) u_next = cross[a];
    double len = u_next - u_cur;
    if (len < 0.0) len = 0.0;
    size_t bin = ((((size_t)it * P.G + p.g) * P.mesh_n[2] + idx[2]) * P.mesh_n[1] + idx[1]) * P.mesh_n[0] + idx[0];
    P.x[bin] += p.w * len;
    u_cur = u_next;
    if (u_next >= u_out) break;
    bool left = false;
    for (int a = 0; a < 3; ++a) {
      if (cross[a] <= u_next) {
        idx[a] += (o[a] > 0.0) ? 1 : -1;
        if (idx[a] < 0 || idx[a] >= P.mesh_n[a]) left = true;
      }
    }
    if (cross[3] <= u_next) { it += 1; if (it >= P.Nt) left = true; }
    if (left) break;
  }
}

// ---------------------------------------------------------------------------------------------
// A.3 source particle of history h
// ---------------------------------------------------------------------------------------------
Particle source_particle(orc_problem &P, uint64_t seed, uint64_t h) {
  Particle p;
  p.key = source_key(seed, h); p.ctr = 0;
  double xi_x = draw(p.key, p.ctr), xi_y = draw(p.key, p.ctr), xi_z = draw(p.key, p.ctr);
  double xi_t = draw(p.key, p.ctr), xi_g = draw(p.key, p.ctr);
  p.x = P.src_lo[0] + xi_x * (P.src_hi[0] - P.src_lo[0]);
  p.y = P.src_lo[1] + xi_y * (P.src_hi[1] - P.src_lo[1]);
  p.z = P.src_lo[2] + xi_z * (P.src_hi[2] - P.src_lo[2]);
  p.t = P.src_t0 + xi_t * (P.src_t1 - P.src_t0);
  p.g = sample_cdf(P.src_pdf.data(), P.G, xi_g);
  if (P.src_dir_mode == 0) {
    double xi_mu = draw(p.key, p.ctr), xi_phi = draw(p.key, p.ctr);
    isotropic(xi_mu, xi_phi, p.ux, p.uy, p.uz);
  } else {
    p.ux = P.src_dir[0]; p.uy = P.src_dir[1]; p.uz = P.src_dir[2];
  }
  p.w = 1.0; p.last_surface = -1; p.alive = true;
  double r[3] = {p.x, p.y, p.z}, o[3] = {p.ux, p.uy, p.uz};
  p.cell = locate(P, r, o, -1);
  p.k = first_census_after(P, p.t);
  P.cnt.source += p.w;
  if (p.cell < 0) { P.cnt.lost += p.w; P.cnt.lost_n += 1; p.alive = false; }
  return p;
}

// A.6 init_child: the child's own stream gives group (chi of the fission-site material) and direction
// (keep_ctr: the birth record has already drawn from its stream -- the generation control of Appendix H)
void init_child(orc_problem &P, Particle &p, bool keep_ctr = false) {
  if (!keep_ctr) p.ctr = 0;
  int m = P.cell_material[p.cell];
  double xi_g = draw(p.key, p.ctr);
  p.g = sample_cdf(&P.chi[(size_t)m * P.G], P.G, xi_g);
  double xi_mu = draw(p.key, p.ctr), xi_phi = draw(p.key, p.ctr);
  isotropic(xi_mu, xi_phi, p.ux, p.uy, p.uz);
  p.last_surface = -1; p.alive = true;
}

inline void bump(orc_problem &P, int which) { if (P.cur_ev) P.cur_ev[which] += 1; }

// ---------------------------------------------------------------------------------------------
// A.5 surface event (post-move).  Returns false when the particle died / was lost.
// ---------------------------------------------------------------------------------------------
void surface_event(orc_problem &P, Particle &p, int s_star) {
  P.cnt.surf_hits += 1; bump(P, 1);
  p.last_surface = s_star;
  const Surface &s = P.surf[s_star];
  if (s.bc == 1) {                                    // vacuum
    P.cnt.leak += p.w; p.alive = false; return;
  }
  if (s.bc == 2) {                                    // reflective: specular about grad f at the hit point
    double g[3]; grad_eval(s, p.x, p.y, p.z, g);
    double norm = std::sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
    double n[3] = {g[0] / norm, g[1] / norm, g[2] / norm};
    double dot = p.ux * n[0] + p.uy * n[1] + p.uz * n[2];
    p.ux = p.ux - 2.0 * dot * n[0];
    p.uy = p.uy - 2.0 * dot * n[1];
    p.uz = p.uz - 2.0 * dot * n[2];
    return;
  }
  double r[3] = {p.x, p.y, p.z}, o[3] = {p.ux, p.uy, p.uz};   // transmission
  int c = locate(P, r, o, s_star);
  if (c < 0) { P.cnt.lost += p.w; P.cnt.lost_n += 1; p.alive = false; return; }
  p.cell = c;
}

// ---------------------------------------------------------------------------------------------
// A.6 collision event.  Children are appended to `bank` as birth records.
// ---------------------------------------------------------------------------------------------
// Appendix I: the collision tally of the paper's Fig. 3 (`add(mcdc.col_tally, part.v, loc2index(part))`),
// read as the collision estimator of the flux: the bin that holds the collision site (r, t, g) takes w / Sigma_t.
// loc2index: i_a = floor((r_a - lo_a) / Delta_a) for lo_a <= r_a < hi_a, largest it with T[it] <= t for
// T[0] <= t < T[Nt]; a site outside the mesh or the time grid scores nothing.
void score_collision(orc_problem &P, const Particle &p, double sig_t) {
  const double r[3] = {p.x, p.y, p.z};
  int idx[3];
  for (int a = 0; a < 3; ++a) {
    if (!(P.mesh_lo[a] <= r[a] && r[a] < P.mesh_hi[a])) return;
    int n = P.mesh_n[a];
    if (n == 1) { idx[a] = 0; continue; }
    double delta = (P.mesh_hi[a] - P.mesh_lo[a]) / (double)n;
    double q = std::floor((r[a] - P.mesh_lo[a]) / delta);
    idx[a] = (q > (double)(n - 1)) ? n - 1 : (int)q;
  }
  if (!(P.T[0] <= p.t && p.t < P.T[P.Nt])) return;
  int it = 0;
  for (int j = 0; j < P.Nt; ++j) if (P.T[j] <= p.t) it = j;
  size_t bin = ((((size_t)it * P.G + p.g) * P.mesh_n[2] + idx[2]) * P.mesh_n[1] + idx[1]) * P.mesh_n[0] + idx[0];
  P.xc[bin] += p.w / sig_t;
}

void collision_event(orc_problem &P, Particle &p, std::deque<BankItem> &bank) {
  P.cnt.collisions += 1; bump(P, 0);
  p.last_surface = -1;
  const int m = P.cell_material[p.cell], G = P.G;
  const size_t mg = (size_t)m * G + p.g;
  if (P.col_on) score_collision(P, p, P.sigma_t[mg]);   // with the weight the particle arrives with
  double xi = draw(p.key, p.ctr);
  double s_tot = P.sigma_s_tot[mg];
  bool scatter;
  if (P.tech.implicit_capture) {
    // G.1 implicit capture: the captured fraction leaves the weight, the reaction is scatter | fission
    double w_c = p.w * (P.sigma_c[mg] / P.sigma_t[mg]);
    P.cnt.capture += w_c;
    p.w -= w_c;
    double s_r = s_tot + P.sigma_f[mg];
    if (!(s_r > 0.0)) {                               // nothing but capture can happen here
      P.cnt.capture += p.w; p.w = 0.0; p.alive = false; return;
    }
    double y = xi * s_r;
    scatter = (y < s_tot) || P.sigma_f[mg] == 0.0;
  } else {
    double y = xi * P.sigma_t[mg];
    scatter = y < s_tot;
    if (!scatter && (y < s_tot + P.sigma_c[mg] || P.sigma_f[mg] == 0.0)) {   // capture (Sigma_f == 0 falls through to capture)
      P.cnt.capture += p.w; p.alive = false; return;
    }
  }
  if (scatter) {
    // G.2 weight roulette of the surviving particle, before its outgoing flight is sampled
    if (P.tech.wr_threshold > 0.0 && p.w < P.tech.wr_threshold) {
      double xi_r = draw(p.key, p.ctr);
      if (xi_r * P.tech.wr_survive < p.w) { P.cnt.vr_gain += P.tech.wr_survive - p.w; p.w = P.tech.wr_survive; }
      else { P.cnt.vr_loss += p.w; p.alive = false; return; }
    }
    double xi_g = draw(p.key, p.ctr);
    int gp = sample_cdf(&P.sigma_s[mg * G], G, xi_g * s_tot);
    double xi_mu = draw(p.key, p.ctr), xi_phi = draw(p.key, p.ctr);
    isotropic(xi_mu, xi_phi, p.ux, p.uy, p.uz);
    p.g = gp;
    return;
  }
  double xi_nu = draw(p.key, p.ctr);                  // fission
  int n = (int)std::floor(P.nu[mg] + xi_nu);
  P.cnt.fission_abs += p.w;
  P.cnt.production += (double)n * p.w;
  P.cnt.children += (uint64_t)n;
  if (P.cur_ev) P.cur_ev[2] += (uint32_t)n;
  uint32_t c0 = p.ctr;
  for (int j = 0; j < n; ++j) {
    BankItem b; b.is_birth = true;
    b.p = p;
    b.p.key = child_key(p.key, c0, (uint32_t)j);
    b.p.ctr = 0;
    bank.push_back(b);
  }
  p.alive = false;
}

// A.8 census event
void census_event(orc_problem &P, Particle &p, double d) {
  P.cnt.census_events += 1; bump(P, 3);
  P.pop_w[p.k] += p.w; P.pop_n[p.k] += 1;
  if (d > 0.0) p.last_surface = -1;
  if (p.k == P.K - 1) { P.cnt.census_final += p.w; p.alive = false; return; }
  p.k += 1;
}

// A.2 transport one particle until it dies -- or, with stop_at_census (G.3), until it has had a census event
// that left it alive (the particle then waits in the census bank of its batch)
bool transport(orc_problem &P, Particle &p, std::deque<BankItem> &bank, bool stop_at_census = false) {
  while (p.alive) {
    const int m = P.cell_material[p.cell];
    const double sig_t = P.sigma_t[(size_t)m * P.G + p.g];
    const double v = P.speed[p.g];
    double xi = draw(p.key, p.ctr);                   // always consumed (D3)
    double d_coll = (sig_t > 0.0) ? -std::log(xi) / sig_t : INF;
    double d_surf = INF; int s_star = -1;             // A.4 nearest surface: strict '<' in list order
    {
      double r[3] = {p.x, p.y, p.z}, o[3] = {p.ux, p.uy, p.uz};
      for (int i = P.cell_offset[p.cell]; i < P.cell_offset[p.cell + 1]; ++i) {
        int s = P.hs_surface[i];
        double u = surface_distance(P.surf[s], r, o, s == p.last_surface);
        if (u < d_surf) { d_surf = u; s_star = s; }
      }
    }
    double d_time = v * (P.census[p.k] - p.t);
    int ev; double d;                                 // 0 census, 1 surface, 2 collision (D5 priority)
    if (d_time <= d_surf && d_time <= d_coll) { ev = 0; d = d_time; }
    else if (d_surf <= d_coll)               { ev = 1; d = d_surf; }
    else                                     { ev = 2; d = d_coll; }
    score_track(P, p, d);                             // uses pre-move r, t
    p.x += d * p.ux; p.y += d * p.uy; p.z += d * p.uz;
    p.t = (ev == 0) ? P.census[p.k] : p.t + d / v;
    P.cnt.segments += 1;
    if (ev == 0) { census_event(P, p, d); if (stop_at_census && p.alive) return true; }
    else if (ev == 1) surface_event(P, p, s_star);
    else collision_event(P, p, bank);
  }
  return false;
}

// G.3 population control of one batch's census bank at census k: splitting-roulette to the weight
// w_t = W / target.  W is summed in 2^-40 fixed point so that it does not depend on the order of the bank.
// `owner` (the local history index a particle descends from) rides along for the per-history event counts.
const double FIX40 = 1099511627776.0;   // 2^40
typedef std::pair<uint64_t, Particle> Owned;
void population_control(orc_problem &P, const std::vector<Owned> &arrived, uint64_t target, int k,
                        std::vector<Owned> &out, double w_out = 0.0) {   // w_out > 0: weight given to the copies (H.3)
  uint64_t w_fix = 0;
  for (const Owned &a : arrived) w_fix += (uint64_t)(a.second.w * FIX40);
  if (w_fix == 0 || target == 0) return;
  const double w_t = ((double)w_fix / FIX40) / (double)target;
  for (const Owned &a : arrived) {
    Particle q = a.second;
    double xi = draw(q.key, q.ctr);                   // the particle's own stream
    int n = (int)std::floor(q.w / w_t + xi);
    double dw = (double)n * w_t - q.w;
    if (dw > 0.0) P.cnt.vr_gain += dw; else P.cnt.vr_loss += -dw;
    if (n == 0) { P.cnt.pc_removed += 1; continue; }
    P.cnt.pc_added += (uint64_t)(n - 1);
    uint32_t c0 = q.ctr;
    for (int j = 0; j < n; ++j) {
      Particle c = q;                                 // same r, Omega, t, g, cell, last_surface, k
      c.w = (w_out > 0.0) ? w_out : w_t;
      if (j > 0) { c.key = child_key(q.key, c0, (uint32_t)j); c.ctr = 0; }
      out.emplace_back(a.first, c);
      P.pop_w_after[k] += c.w; P.pop_n_after[k] += 1;
    }
  }
}

void close_batch(orc_problem &P) {                    // A.9
  for (size_t i = 0; i < P.n_bins; ++i) {
    double s = P.x[i];
    P.sum[i] += s; P.sumsq[i] += s * s; P.x[i] = 0.0;
  }
  if (P.col_on)
    for (size_t i = 0; i < P.n_bins; ++i) {
      double s = P.xc[i];
      P.sumc[i] += s; P.sumsqc[i] += s * s; P.xc[i] = 0.0;
    }
  P.cnt.batches += 1;
}

void build_boxes(orc_problem &P) {
  // loose axis-aligned culling boxes from a cell's own axis-aligned planes and z/x/y-cylinders or
  // spheres with sense -1; anything else leaves the box unbounded.  Expanded so that a point within
  // rounding of a bounding surface is never culled (the exact half-space test then decides).
  P.bb_lo.assign((size_t)3 * P.C, -INF); P.bb_hi.assign((size_t)3 * P.C, INF);
  for (int c = 0; c < P.C; ++c) {
    if (!P.rgn_off.empty() && P.rgn_off[c] < P.rgn_off[c + 1]) continue;   // a general region: no culling box
    for (int i = P.cell_offset[c]; i < P.cell_offset[c + 1]; ++i) {
      const Surface &s = P.surf[P.hs_surface[i]]; int sense = P.hs_sense[i];
      bool quad = s.A != 0 || s.B != 0 || s.C != 0 || s.D != 0 || s.E != 0 || s.F != 0;
      if (!quad) {
        double lin[3] = {s.G, s.H, s.I};
        int nz = 0, ax = -1;
        for (int a = 0; a < 3; ++a) if (lin[a] != 0.0) { nz++; ax = a; }
        if (nz != 1) continue;
        double pos = -s.J / lin[ax];
        bool upper = (lin[ax] > 0.0) == (sense < 0);   // f<0 with positive slope => coordinate < pos
        if (upper) { if (pos < P.bb_hi[3 * c + ax]) P.bb_hi[3 * c + ax] = pos; }
        else       { if (pos > P.bb_lo[3 * c + ax]) P.bb_lo[3 * c + ax] = pos; }
      } else if (sense < 0 && s.D == 0 && s.E == 0 && s.F == 0 && s.A >= 0 && s.B >= 0 && s.C >= 0) {
        double q[3] = {s.A, s.B, s.C}, lin[3] = {s.G, s.H, s.I};
        // f = sum q_a (r_a - c_a)^2 - R2 with c_a = -lin_a / (2 q_a); R2 = sum q_a c_a^2 - J
        double R2 = -s.J, cen[3] = {0, 0, 0};
        for (int a = 0; a < 3; ++a) if (q[a] > 0.0) { cen[a] = -lin[a] / (2.0 * q[a]); R2 += q[a] * cen[a] * cen[a]; }
        bool ok = R2 > 0.0;
        for (int a = 0; a < 3; ++a) if (q[a] == 0.0 && lin[a] != 0.0) ok = false;
        if (!ok) continue;
        for (int a = 0; a < 3; ++a) if (q[a] > 0.0) {
          double h = std::sqrt(R2 / q[a]);
          if (cen[a] - h > P.bb_lo[3 * c + a]) P.bb_lo[3 * c + a] = cen[a] - h;
          if (cen[a] + h < P.bb_hi[3 * c + a]) P.bb_hi[3 * c + a] = cen[a] + h;
        }
      }
    }
    for (int a = 0; a < 3; ++a) {
      double lo = P.bb_lo[3 * c + a], hi = P.bb_hi[3 * c + a];
      double pad = 1e-6 * (1.0 + std::fabs(lo == -INF ? 0.0 : lo) + std::fabs(hi == INF ? 0.0 : hi));
      P.bb_lo[3 * c + a] = lo - pad; P.bb_hi[3 * c + a] = hi + pad;
    }
  }
}

}  // namespace

// =============================================================================================
// C interface
// =============================================================================================
extern "C" {

int orc_create(const orc_desc *d, orc_problem **out) {
  if (!d || !out) return -1;
  if (d->G < 1 || d->M < 1 || d->S < 1 || d->C < 1 || d->Nt < 1 || d->K < 1) return -1;
  orc_problem *P = new orc_problem();
  P->G = d->G; P->M = d->M; P->S = d->S; P->C = d->C;
  size_t MG = (size_t)d->M * d->G;
  P->sigma_t.assign(d->sigma_t, d->sigma_t + MG);
  P->sigma_c.assign(d->sigma_c, d->sigma_c + MG);
  P->sigma_f.assign(d->sigma_f, d->sigma_f + MG);
  P->nu.assign(d->nu, d->nu + MG);
  P->chi.assign(d->chi, d->chi + MG);
  P->sigma_s.assign(d->sigma_s, d->sigma_s + MG * d->G);
  P->speed.assign(d->speed, d->speed + d->G);
  P->sigma_s_tot.assign(MG, 0.0);
  for (size_t mg = 0; mg < MG; ++mg) {               // summed in increasing g' (A.1)
    double s = 0.0;
    for (int gp = 0; gp < d->G; ++gp) s += P->sigma_s[mg * d->G + gp];
    P->sigma_s_tot[mg] = s;
  }
  P->surf.resize(d->S);
  for (int s = 0; s < d->S; ++s) {
    const double *c = d->surf_coef + (size_t)10 * s;
    Surface &q = P->surf[s];
    q.A = c[0]; q.B = c[1]; q.C = c[2]; q.D = c[3]; q.E = c[4]; q.F = c[5]; q.G = c[6]; q.H = c[7]; q.I = c[8]; q.J = c[9];
    q.bc = d->surf_bc[s];
  }
  P->cell_offset.assign(d->cell_offset, d->cell_offset + d->C + 1);
  int nhs = P->cell_offset[d->C];
  P->hs_surface.assign(d->hs_surface, d->hs_surface + nhs);
  P->hs_sense.assign(d->hs_sense, d->hs_sense + nhs);
  P->cell_material.assign(d->cell_material, d->cell_material + d->C);
  for (int a = 0; a < 3; ++a) {
    P->src_lo[a] = d->src_lo[a]; P->src_hi[a] = d->src_hi[a]; P->src_dir[a] = d->src_dir[a];
    P->mesh_lo[a] = d->mesh_lo[a]; P->mesh_hi[a] = d->mesh_hi[a]; P->mesh_n[a] = d->mesh_n[a];
    if (d->mesh_n[a] < 1) { delete P; return -1; }
  }
  P->src_t0 = d->src_t0; P->src_t1 = d->src_t1; P->src_dir_mode = d->src_dir_mode;
  P->src_pdf.assign(d->src_group_pdf, d->src_group_pdf + d->G);
  P->Nt = d->Nt; P->T.assign(d->time_edges, d->time_edges + d->Nt + 1);
  P->K = d->K; P->census.assign(d->census, d->census + d->K);
  P->n_bins = (size_t)d->Nt * d->G * d->mesh_n[2] * d->mesh_n[1] * d->mesh_n[0];
  build_boxes(*P);
  P->cur_ev = nullptr;
  std::memset(&P->tech, 0, sizeof(P->tech));
  P->col_on = 0;
  orc_reset(P);
  *out = P;
  return 0;
}

// Appendix J: general CSG regions; validates the postfix expressions (operands in range, stack never underflows,
// exactly one value left).  NULL pointers: every cell is the plain intersection again.
int orc_regions_set(orc_problem *P, const int32_t *region_offset, const int32_t *region_rpn) {
  if (!P) return -1;
  P->rgn_off.clear(); P->rgn_tok.clear();
  if (region_offset && region_rpn) {
    for (int c = 0; c < P->C; ++c) {
      int depth = 0;
      const int nh = P->cell_offset[c + 1] - P->cell_offset[c];
      if (region_offset[c + 1] < region_offset[c]) return -3;
      for (int k = region_offset[c]; k < region_offset[c + 1]; ++k) {
        int t = region_rpn[k];
        if (t >= 0) { if (t >= nh) return -3; depth += 1; }
        else if (t == -3) { if (depth < 1) return -3; }
        else if (t == -1 || t == -2) { if (depth < 2) return -3; depth -= 1; }
        else return -3;
      }
      if (region_offset[c + 1] > region_offset[c] && depth != 1) return -3;
    }
    P->rgn_off.assign(region_offset, region_offset + P->C + 1);
    P->rgn_tok.assign(region_rpn, region_rpn + region_offset[P->C]);
  }
  build_boxes(*P);
  return 0;
}

int orc_technique_set(orc_problem *P, const orc_technique *t) {
  if (!P) return -1;
  if (!t) { std::memset(&P->tech, 0, sizeof(P->tech)); return 0; }
  if (t->wr_threshold > 0.0 && !(t->wr_survive >= t->wr_threshold)) return -1;
  P->tech = *t;
  return 0;
}

int orc_census_after_get(const orc_problem *P, double *w, uint64_t *n, size_t K) {
  if (K != (size_t)P->K) return -4;
  for (size_t k = 0; k < K; ++k) { w[k] = P->pop_w_after[k]; n[k] = P->pop_n_after[k]; }
  return 0;
}

// unit-level: the control applied to a bank given as arrays (pins of G.3); n_out[i] = copies of particle i
int orc_population_control(orc_problem *P, size_t n, const double *w, const uint64_t *key, const uint32_t *ctr,
                           uint64_t target, int32_t *n_out, double *w_t_out) {
  std::vector<Owned> in, out;
  for (size_t i = 0; i < n; ++i) {
    Particle q; std::memset(&q, 0, sizeof(q));
    q.w = w[i]; q.key = key[i]; q.ctr = ctr[i]; q.alive = true;
    in.emplace_back((uint64_t)i, q);
  }
  orc_counters save = P->cnt;
  std::vector<double> sw = P->pop_w_after; std::vector<uint64_t> sn = P->pop_n_after;
  population_control(*P, in, target, 0, out);
  P->cnt = save; P->pop_w_after = sw; P->pop_n_after = sn;
  for (size_t i = 0; i < n; ++i) n_out[i] = 0;
  for (const Owned &o : out) n_out[o.first] += 1;
  *w_t_out = out.empty() ? 0.0 : out[0].second.w;
  return 0;
}

void orc_destroy(orc_problem *p) { delete p; }

void orc_reset(orc_problem *P) {
  P->x.assign(P->n_bins, 0.0); P->sum.assign(P->n_bins, 0.0); P->sumsq.assign(P->n_bins, 0.0);
  P->xc.assign(P->n_bins, 0.0); P->sumc.assign(P->n_bins, 0.0); P->sumsqc.assign(P->n_bins, 0.0);
  P->pop_w.assign(P->K, 0.0); P->pop_n.assign(P->K, 0);
  P->pop_w_after.assign(P->K, 0.0); P->pop_n_after.assign(P->K, 0);
  std::memset(&P->cnt, 0, sizeof(P->cnt));
  P->batch_size = 0; P->hist_ev.clear(); P->cur_ev = nullptr;
}

// A.2 + A.9: histories first..first+N-1 in B batches of N/B
int orc_run(orc_problem *P, uint64_t n_histories, uint64_t seed, const orc_run_opts *o) {
  orc_run_opts def = {1u, 0ull, 0, 0, 0};
  if (!o) o = &def;
  uint32_t B = o->n_batches ? o->n_batches : 1u;
  if (n_histories == 0 || n_histories % B != 0) return -1;
  uint64_t hb = n_histories / B;
  if (P->batch_size != 0 && P->batch_size != hb) return -1;
  P->batch_size = hb;
  if (o->record_history_events) P->hist_ev.assign((size_t)n_histories * 4, 0u); else P->hist_ev.clear();
  std::deque<BankItem> bank;
  if (P->tech.population_control) {
    // G.3: batch-synchronous census steps.  Step k transports every particle whose next census is C[k]
    // (sources born in the step, survivors of the control at C[k-1], and all their fission progeny) up to
    // C[k]; the arrivals are controlled and become the live bank of step k+1.
    const uint64_t target = P->tech.pc_target ? P->tech.pc_target : hb;
    for (uint32_t b = 0; b < B; ++b) {
      std::vector<Owned> src;                              // (local history index, particle) of the batch
      for (uint64_t i = 0; i < hb; ++i) {
        uint64_t local = (uint64_t)b * hb + (o->reverse_histories ? (hb - 1 - i) : i);
        P->cnt.histories += 1;
        Particle p = source_particle(*P, seed, o->first_history_id + local);
        if (p.alive) src.emplace_back(local, p);
      }
      std::vector<Owned> live, arrived;
      for (int k = 0; k < P->K; ++k) {
        for (auto &sp : src) if (sp.second.k == k) live.push_back(sp);
        arrived.clear();
        for (auto &lp : live) {
          P->cur_ev = o->record_history_events ? &P->hist_ev[(size_t)lp.first * 4] : nullptr;
          BankItem first; first.is_birth = false; first.p = lp.second;
          bank.push_back(first);
          while (!bank.empty()) {
            BankItem it;
            if (o->bank_fifo) { it = bank.front(); bank.pop_front(); }
            else              { it = bank.back();  bank.pop_back(); }
            if (it.is_birth) init_child(*P, it.p);
            if (transport(*P, it.p, bank, true)) arrived.emplace_back(lp.first, it.p);
          }
        }
        live.clear();
        if (k == P->K - 1) break;
        population_control(*P, arrived, target, k, live);
      }
      close_batch(*P);
    }
    P->cur_ev = nullptr;
    return 0;
  }
  for (uint32_t b = 0; b < B; ++b) {
    for (uint64_t i = 0; i < hb; ++i) {
      uint64_t local = (uint64_t)b * hb + (o->reverse_histories ? (hb - 1 - i) : i);
      uint64_t h = o->first_history_id + local;
      P->cur_ev = o->record_history_events ? &P->hist_ev[(size_t)local * 4] : nullptr;
      P->cnt.histories += 1;
      BankItem src; src.is_birth = false; src.p = source_particle(*P, seed, h);
      if (src.p.alive) bank.push_back(src);
      while (!bank.empty()) {
        BankItem it;
        if (o->bank_fifo) { it = bank.front(); bank.pop_front(); }
        else              { it = bank.back();  bank.pop_back(); }
        if (it.is_birth) init_child(*P, it.p);
        transport(*P, it.p, bank);
      }
    }
    close_batch(*P);
  }
  P->cur_ev = nullptr;
  return 0;
}

// ---------------------------------------------------------------------------------------------
// Appendix H of DESIGN.md: k-eigenvalue mode, power iteration over fission generations.
//  H.1 generation 0 = the problem's source, N histories of weight 1; a generation transports its particles
//      until they die; fission children are NOT transported in the generation that made them, they are its
//      fission bank.  k_g = (weight of the children made in generation g) / (weight that started it).
//  H.2 tallies: every generation from n_inactive on is one statistical batch of N histories; earlier ones
//      are discarded.
//  H.3 the next generation = the population control of G.3 applied to the fission bank (target N, every
//      birth record draws xi from its own stream at counter 0), the copies taking weight 1; init_child then
//      goes on from the record's counter.
// ---------------------------------------------------------------------------------------------
int orc_run_eigenvalue(orc_problem *P, uint64_t N, uint64_t seed, uint32_t n_inactive, uint32_t n_active,
                       int32_t reverse_order, double *k_gen) {
  if (!P || !k_gen || N == 0 || n_active == 0) return -1;
  if (P->batch_size != 0 && P->batch_size != N) return -1;
  P->batch_size = N;
  P->hist_ev.clear(); P->cur_ev = nullptr;
  std::vector<Owned> cur, next;                           // (is_birth flag in .first, particle)
  for (uint64_t h = 0; h < N; ++h) {
    Particle p = source_particle(*P, seed, h);
    if (p.alive) cur.emplace_back(0u, p);
  }
  const uint32_t G_total = n_inactive + n_active;
  std::deque<BankItem> fis;
  for (uint32_t g = 0; g < G_total; ++g) {
    double start_w = 0.0;
    for (const Owned &c : cur) start_w += c.second.w;
    const double prod0 = P->cnt.production;
    fis.clear();
    for (size_t i = 0; i < cur.size(); ++i) {
      Owned &c = cur[reverse_order ? cur.size() - 1 - i : i];
      Particle p = c.second;
      if (c.first) init_child(*P, p, true);
      transport(*P, p, fis);                              // children pile up in fis, nobody pops them here
    }
    k_gen[g] = start_w > 0.0 ? (P->cnt.production - prod0) / start_w : 0.0;
    if (g >= n_inactive) { P->cnt.histories += N; close_batch(*P); }
    else { std::fill(P->x.begin(), P->x.end(), 0.0); std::fill(P->xc.begin(), P->xc.end(), 0.0); }
    if (g + 1 == G_total) break;                          // the last generation's bank is not needed
    std::vector<Owned> bank;
    for (const BankItem &b : fis) bank.emplace_back(1u, b.p);
    next.clear();
    population_control(*P, bank, N, 0, next, 1.0);
    cur.swap(next);
    if (cur.empty()) { for (uint32_t r = g + 1; r < G_total; ++r) k_gen[r] = 0.0; break; }
  }
  return 0;
}

int orc_tally_sums_get(const orc_problem *P, double *sum, double *sumsq, size_t n_bins) {
  if (n_bins != P->n_bins) return -4;
  std::memcpy(sum, P->sum.data(), n_bins * sizeof(double));
  std::memcpy(sumsq, P->sumsq.data(), n_bins * sizeof(double));
  return 0;
}

// A.9: mean = sum / N; m_b = S_b * B / N; sdev = sqrt((sum m_b^2 / B - mean^2) / (B - 1)); B = 1 -> 0
int orc_tallies_get(const orc_problem *P, double *mean, double *sdev, size_t n_bins) {
  if (n_bins != P->n_bins) return -4;
  double N = (double)P->cnt.histories, B = (double)P->cnt.batches;
  if (N == 0.0) return -1;
  double hb = N / B;
  for (size_t i = 0; i < n_bins; ++i) {
    double mu = P->sum[i] / N;
    mean[i] = mu;
    if (B > 1.0) {
      double m2 = P->sumsq[i] / (hb * hb) / B;
      double var = (m2 - mu * mu) / (B - 1.0);
      sdev[i] = var > 0.0 ? std::sqrt(var) : 0.0;
    } else sdev[i] = 0.0;
  }
  return 0;
}

int orc_collision_tally_enable(orc_problem *P, int on) { if (!P) return -1; P->col_on = on ? 1 : 0; return 0; }

// same statistics as orc_tallies_get (A.9), from the collision-estimator accumulators
int orc_collision_tallies_get(const orc_problem *P, double *mean, double *sdev, size_t n_bins) {
  if (n_bins != P->n_bins) return -4;
  double N = (double)P->cnt.histories, B = (double)P->cnt.batches;
  if (N == 0.0) return -1;
  double hb = N / B;
  for (size_t i = 0; i < n_bins; ++i) {
    double mu = P->sumc[i] / N;
    mean[i] = mu;
    if (B > 1.0) {
      double m2 = P->sumsqc[i] / (hb * hb) / B;
      double var = (m2 - mu * mu) / (B - 1.0);
      sdev[i] = var > 0.0 ? std::sqrt(var) : 0.0;
    } else sdev[i] = 0.0;
  }
  return 0;
}

int orc_counters_get(const orc_problem *P, orc_counters *c) { *c = P->cnt; return 0; }

int orc_census_get(const orc_problem *P, double *pop_w, uint64_t *pop_n, size_t K) {
  if (K != (size_t)P->K) return -4;
  for (size_t k = 0; k < K; ++k) { pop_w[k] = P->pop_w[k]; pop_n[k] = P->pop_n[k]; }
  return 0;
}

int orc_history_events_get(const orc_problem *P, uint32_t *ev, size_t n) {
  if (n * 4 != P->hist_ev.size()) return -4;
  std::memcpy(ev, P->hist_ev.data(), P->hist_ev.size() * sizeof(uint32_t));
  return 0;
}

uint64_t orc_mix64(uint64_t z) { return mix64(z); }
uint64_t orc_source_key(uint64_t seed, uint64_t h) { return source_key(seed, h); }
uint64_t orc_child_key(uint64_t kp, uint32_t c0, uint32_t j) { return child_key(kp, c0, j); }
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox4x32_10(ctr, key, out); }
void orc_draws(uint64_t key, uint32_t first_ctr, size_t n, double *out) {
  uint32_t c = first_ctr;
  for (size_t i = 0; i < n; ++i) out[i] = draw(key, c);
}
double orc_surface_distance(const double coef[10], const double r[3], const double omega[3], int on_surface) {
  Surface s = {coef[0], coef[1], coef[2], coef[3], coef[4], coef[5], coef[6], coef[7], coef[8], coef[9], 0};
  return surface_distance(s, r, omega, on_surface != 0);
}
int orc_locate(const orc_problem *P, const double r[3], const double omega[3]) { return locate(*P, r, omega, -1); }

int orc_stream(const orc_problem *P0, double r[3], double omega[3], int32_t *cell, int max_events) {
  orc_problem &P = *const_cast<orc_problem *>(P0);
  orc_counters save = P.cnt;
  Particle p; p.x = r[0]; p.y = r[1]; p.z = r[2]; p.ux = omega[0]; p.uy = omega[1]; p.uz = omega[2];
  p.t = 0; p.w = 1; p.g = 0; p.cell = *cell; p.last_surface = -1; p.key = 0; p.ctr = 0; p.k = 0; p.alive = true;
  int n = 0;
  while (p.alive && n < max_events) {
    double d_surf = INF; int s_star = -1;
    double rr[3] = {p.x, p.y, p.z}, oo[3] = {p.ux, p.uy, p.uz};
    for (int i = P.cell_offset[p.cell]; i < P.cell_offset[p.cell + 1]; ++i) {
      int s = P.hs_surface[i];
      double u = surface_distance(P.surf[s], rr, oo, s == p.last_surface);
      if (u < d_surf) { d_surf = u; s_star = s; }
    }
    if (s_star < 0) break;
    p.x += d_surf * p.ux; p.y += d_surf * p.uy; p.z += d_surf * p.uz;
    surface_event(P, p, s_star);
    n += 1;
  }
  P.cnt = save;
  r[0] = p.x; r[1] = p.y; r[2] = p.z; omega[0] = p.ux; omega[1] = p.uy; omega[2] = p.uz;
  *cell = p.alive ? p.cell : -1;
  return n;
}

int orc_score_segment(orc_problem *P, const double r[3], const double omega[3], double t, int g, double w, double d) {
  if (g < 0 || g >= P->G) return -1;
  Particle p; p.x = r[0]; p.y = r[1]; p.z = r[2]; p.ux = omega[0]; p.uy = omega[1]; p.uz = omega[2];
  p.t = t; p.w = w; p.g = g; p.cell = 0; p.last_surface = -1; p.key = 0; p.ctr = 0; p.k = 0; p.alive = true;
  score_track(*P, p, d);
  return 0;
}

int orc_close_batch(orc_problem *P, uint64_t histories_in_batch) {
  if (P->batch_size != 0 && P->batch_size != histories_in_batch) return -1;
  P->batch_size = histories_in_batch;
  P->cnt.histories += histories_in_batch;
  close_batch(*P);
  return 0;
}

}  // extern "C"
