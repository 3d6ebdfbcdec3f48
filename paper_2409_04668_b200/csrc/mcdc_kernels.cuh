// mcdc_kernels.cuh -- source, transport and close-out kernels (sm_100a).
//
// Scheduler (replaces the paper's Harmonize runtime): one persistent grid per census
// step.  A block adopts one statistical-batch slot at a time; its warps refill idle lanes from the
// slot's bank cursor with a ballot-aggregated atomic, keep the particle state in registers from
// segment to segment, and hand finished particles to the census bank / fission bank with
// ballot-aggregated appends.  Track-length scores go to a shared-memory copy of the step's tally slab
// (match_any-aggregated when few bins are hit) and are flushed with fp64 RED to the slot's accumulator.
#pragma once
#include "mcdc_device.cuh"

namespace mcdc {

constexpr int TRANSPORT_THREADS = 256;

// ------------------------------------------------------------------------------------------------
// small warp helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(MCDC_FULL, v, o);
  return v;
}

// ballot-aggregated append: lanes with `want` get consecutive indices from *counter
__device__ __forceinline__ uint32_t warp_append(uint32_t *counter, bool want) {
  unsigned m = __ballot_sync(MCDC_FULL, want);
  if (m == 0u) return 0u;
  int leader = __ffs(m) - 1;
  uint32_t base = 0u;
  if (lane_id() == leader) base = atomicAdd(counter, (uint32_t)__popc(m));
  base = __shfl_sync(MCDC_FULL, base, leader);
  return base + (uint32_t)__popc(m & ((1u << lane_id()) - 1u));
}

// ------------------------------------------------------------------------------------------------
// Tally sink: shared-memory slab (privatised) or the slot's global accumulator.
// Called warp-converged; bin < 0 means "nothing to add for this lane".
// ------------------------------------------------------------------------------------------------
struct TallySink {
  double *slab;      // shared memory, or nullptr
  double *global_x;  // slot accumulator x[slot][n_bins]
  long long slab_lo; // first global bin held by the slab
  int slab_bins;
};

__device__ __forceinline__ void tally_add_converged(const TallySink &S, long long bin, double val) {
  unsigned valid = __ballot_sync(MCDC_FULL, bin >= 0);
  if (valid == 0u) return;
  if (S.slab != nullptr) {
    long long rel = bin - S.slab_lo;
    if (bin >= 0 && (rel < 0 || rel >= S.slab_bins)) {     // outside the step's slab (rounding-length pieces)
      atomicAdd(S.global_x + bin, val);
      bin = -1;
    }
    int b = (bin >= 0) ? (int)rel : -1;
    unsigned peers = __match_any_sync(MCDC_FULL, b);
    unsigned leaders = __ballot_sync(MCDC_FULL, b >= 0 && lane_id() == __ffs(peers) - 1);
    if (__popc(leaders) <= 3) {
      while (leaders) {
        int l = __ffs(leaders) - 1;
        leaders &= leaders - 1u;
        int lb = __shfl_sync(MCDC_FULL, b, l);
        double v = warp_sum((b == lb) ? val : 0.0);
        if (lane_id() == l) atomicAdd(S.slab + lb, v);
      }
    } else if (b >= 0) {
      atomicAdd(S.slab + b, val);
    }
  } else if (bin >= 0) {
    atomicAdd(S.global_x + bin, val);
  }
}

// ------------------------------------------------------------------------------------------------
// A.7 track-length scoring: 4-D DDA from the pre-move state.  Warp-converged: every lane calls it,
// lanes without a segment pass active = false.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void score_track(const Tables &T, const TallySink &S, bool active, double x, double y,
                                            double z, double ux, double uy, double uz, double t, double w, int g,
                                            double d) {
  const double INF = CUDART_INF;
  const double r[3] = {x, y, z}, o[3] = {ux, uy, uz};
  double inv_o[3];
  double u_in = 0.0, u_out = d, u_cur = 0.0;
  int idx[3] = {0, 0, 0};
  int it = 0;
  double v = 0.0;
  bool more = active;
  if (more) {
    v = __ldg(T.speed + g);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double lo = T.mesh_lo[a], hi = T.mesh_hi[a];
      if (o[a] == 0.0) {
        inv_o[a] = INF;
        if (!(lo <= r[a] && r[a] < hi)) more = false;
      } else {
        inv_o[a] = 1.0 / o[a];
        double u0 = (lo - r[a]) * inv_o[a], u1 = (hi - r[a]) * inv_o[a];
        if (o[a] < 0.0) { double tmp = u0; u0 = u1; u1 = tmp; }
        u_in = fmax(u_in, u0); u_out = fmin(u_out, u1);
      }
    }
    u_in = fmax(u_in, (__ldg(T.T) - t) * v);
    u_out = fmin(u_out, (__ldg(T.T + T.Nt) - t) * v);
    if (!(u_in < u_out)) more = false;
  }
  if (more) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const int n = T.mesh_n[a];
      if (n > 1) {
        double q = floor((r[a] + u_in * o[a] - T.mesh_lo[a]) * T.mesh_inv_d[a]);
        idx[a] = (q < 0.0) ? 0 : ((q > (double)(n - 1)) ? n - 1 : (int)q);
      }
    }
    const double t_in = t + u_in * __ldg(T.inv_speed + g);
    // largest it with T[it] <= t_in (binary search over the edge array)
    int lo = 0, hi = T.Nt - 1;
    while (lo < hi) {
      int mid = (lo + hi + 1) >> 1;
      if (__ldg(T.T + mid) <= t_in) lo = mid; else hi = mid - 1;
    }
    it = lo;
    u_cur = u_in;
  }
  while (__any_sync(MCDC_FULL, more)) {
    long long bin = -1;
    double val = 0.0;
    if (more) {
      double cross[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        if (o[a] == 0.0) { cross[a] = INF; continue; }
        double edge;
        if (T.mesh_n[a] == 1) edge = (o[a] > 0.0) ? T.mesh_hi[a] : T.mesh_lo[a];
        else edge = T.mesh_lo[a] + (double)(idx[a] + (o[a] > 0.0 ? 1 : 0)) * T.mesh_d[a];
        cross[a] = (edge - r[a]) * inv_o[a];
      }
      const double cross_t = (__ldg(T.T + it + 1) - t) * v;
      double u_next = fmin(fmin(u_out, cross_t), fmin(cross[0], fmin(cross[1], cross[2])));
      bin = ((((long long)it * T.G + g) * T.mesh_n[2] + idx[2]) * T.mesh_n[1] + idx[1]) * T.mesh_n[0] + idx[0];
      val = w * fmax(u_next - u_cur, 0.0);
      u_cur = u_next;
      if (u_next >= u_out) more = false;
      else {
#pragma unroll
        for (int a = 0; a < 3; ++a)
          if (cross[a] <= u_next) {
            idx[a] += (o[a] > 0.0) ? 1 : -1;
            if (idx[a] < 0 || idx[a] >= T.mesh_n[a]) more = false;
          }
        if (cross_t <= u_next) { it += 1; if (it >= T.Nt) more = false; }
      }
    }
    tally_add_converged(S, bin, val);
  }
}

// ------------------------------------------------------------------------------------------------
// match_any-aggregated append for lanes that may target different slots (source kernel)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t warp_append_by_slot(uint32_t *counters, int slot) {
  unsigned peers = __match_any_sync(MCDC_FULL, slot);
  int leader = __ffs(peers) - 1;
  uint32_t base = 0u;
  if (slot >= 0 && lane_id() == leader) base = atomicAdd(counters + slot, (uint32_t)__popc(peers));
  base = __shfl_sync(MCDC_FULL, base, leader);
  return base + (uint32_t)__popc(peers & ((1u << lane_id()) - 1u));
}

// block-wide sum of per-thread doubles into one global atomic (blockDim.x <= 1024)
__device__ __forceinline__ void block_atomic_add(double *dst, double v, double *scratch /* [32] shared */) {
  v = warp_sum(v);
  if (lane_id() == 0) scratch[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x < 32) {
    double s = (threadIdx.x < (blockDim.x + 31) / 32) ? scratch[threadIdx.x] : 0.0;
    s = warp_sum(s);
    if (threadIdx.x == 0 && s != 0.0) atomicAdd(dst, s);
  }
  __syncthreads();
}
__device__ __forceinline__ void block_atomic_add_u64(unsigned long long *dst, unsigned long long v,
                                                     unsigned long long *scratch /* [32] shared */) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(MCDC_FULL, v, o);
  if (lane_id() == 0) scratch[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x < 32) {
    unsigned long long s = (threadIdx.x < (blockDim.x + 31) / 32) ? scratch[threadIdx.x] : 0ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(MCDC_FULL, s, o);
    if (threadIdx.x == 0 && s != 0ull) atomicAdd(dst, s);
  }
  __syncthreads();
}

// ------------------------------------------------------------------------------------------------
// Source kernel (A.3): one thread per history of the sub-batch; histories whose birth time falls
// in census step k are appended to the live bank of their batch slot.
// ------------------------------------------------------------------------------------------------
struct SourceParams {
  unsigned long long seed_mixed;       // M(seed + gamma)
  unsigned long long first_history;    // global id of local history 0 of this sub-batch
  uint32_t n_hist;                     // histories in this sub-batch
  uint32_t hb;                         // histories per slot
  uint32_t cap;
  int k;                               // census step being fed
  int single_step;                     // all sources are born in step k (skip the time filter)
};

__global__ void __launch_bounds__(256) k_source(Tables T, SourceParams P, Bank out, DevCounters *cnt) {
  __shared__ double scratch[32];
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  bool live = i < P.n_hist;
  double x = 0, y = 0, z = 0, ux = 0, uy = 0, uz = 1, t = 0;
  double xi_x = 0, xi_y = 0, xi_z = 0, xi_t = 0;
  int g = 0, cell = -1;
  uint32_t ctr = 0;
  unsigned long long key = 0;
  if (live) {
    key = mix64(P.seed_mixed ^ (P.first_history + i));
    draw2(key, ctr, xi_x, xi_y);
    draw2(key, ctr, xi_z, xi_t);
    t = T.src_t0 + xi_t * (T.src_t1 - T.src_t0);
    if (!P.single_step) {
      int k0 = T.K - 1;                  // smallest k with C[k] > t (last step when none, D15)
      for (int k = 0; k < T.K; ++k)
        if (__ldg(T.census + k) > t) { k0 = k; break; }
      if (k0 != P.k) live = false;
    }
  }
  if (live) {
    double xi_g = draw(key, ctr);
    x = T.src_lo[0] + xi_x * (T.src_hi[0] - T.src_lo[0]);
    y = T.src_lo[1] + xi_y * (T.src_hi[1] - T.src_lo[1]);
    z = T.src_lo[2] + xi_z * (T.src_hi[2] - T.src_lo[2]);
    g = sample_cdf(T.src_cdf, T.G, T.src_last, xi_g);
    if (T.src_dir_mode == 0) {
      double xi_mu, xi_phi;
      draw2(key, ctr, xi_mu, xi_phi);
      isotropic(xi_mu, xi_phi, ux, uy, uz);
    } else {
      ux = T.src_dir[0]; uy = T.src_dir[1]; uz = T.src_dir[2];
    }
    cell = locate_source(T, x, y, z, ux, uy, uz);
  }
  const bool lost = live && cell < 0;
  const bool keep = live && cell >= 0;
  const int slot = keep ? (int)(i / P.hb) : -1;
  uint32_t idx = warp_append_by_slot(out.count, slot);
  if (keep) {
    if (idx >= P.cap) {
      atomicExch(&cnt->overflow, 1);
    } else {
      size_t j = (size_t)slot * P.cap + idx;
      out.x[j] = x; out.y[j] = y; out.z[j] = z;
      out.ux[j] = ux; out.uy[j] = uy; out.uz[j] = uz;
      out.t[j] = t; out.w[j] = 1.0;
      out.key[j] = key;
      out.meta[j] = make_int4(cell, -1, (int)ctr, g);
      out.hid[j] = i;
    }
  }
  block_atomic_add(&cnt->ledger[0], live ? 1.0 : 0.0, scratch);
  block_atomic_add(&cnt->ledger[6], lost ? 1.0 : 0.0, scratch);
  block_atomic_add_u64(&cnt->n[0], live ? 1ull : 0ull, (unsigned long long *)scratch);
  block_atomic_add_u64(&cnt->n[6], lost ? 1ull : 0ull, (unsigned long long *)scratch);
}

// ------------------------------------------------------------------------------------------------
// Transport kernel: one census step (or one fission generation inside it) for every slot.
// ------------------------------------------------------------------------------------------------
enum { LED_PRODUCTION = 0, LED_CAPTURE, LED_FISSION_ABS, LED_LEAK, LED_CENSUS_FINAL, LED_LOST, LED_N };
enum { CNT_COLL = 0, CNT_SURF, CNT_CENSUS, CNT_CHILDREN, CNT_LOST, CNT_N };

struct TransportArgs {
  Bank in, census_out, sec_out;
  double *x_acc;                 // [n_slots][n_bins] batch accumulators
  DevCounters *cnt;
  double *pop_w;                 // [K]
  unsigned long long *pop_n;     // [K]
  uint32_t *ev;                  // [n_hist][4] per-history event counts of this sub-batch, or nullptr
};

__global__ void __launch_bounds__(TRANSPORT_THREADS) k_transport(Tables T, StepParams P, TransportArgs A) {
  extern __shared__ double slab[];                       // [P.slab_bins]
  __shared__ double s_led[LED_N][TRANSPORT_THREADS];
  __shared__ uint32_t s_cnt[CNT_N][TRANSPORT_THREADS];
  __shared__ double s_scratch[32];
  __shared__ int s_flag;
  const double INF = CUDART_INF;
  const int tid = threadIdx.x, lane = tid & 31;
#pragma unroll
  for (int e = 0; e < LED_N; ++e) s_led[e][tid] = 0.0;
#pragma unroll
  for (int e = 0; e < CNT_N; ++e) s_cnt[e][tid] = 0u;
  double popw = 0.0;
  uint32_t popn = 0u;

  for (int probe = 0; probe < P.n_slots; ++probe) {
    const int slot = (int)((blockIdx.x + (unsigned)probe) % (unsigned)P.n_slots);
    const uint32_t n_in = A.in.count[slot];
    if (tid == 0) s_flag = (*(volatile uint32_t *)(A.in.cursor + slot) < n_in) ? 1 : 0;
    __syncthreads();
    const bool has_work = s_flag != 0;
    __syncthreads();
    if (!has_work) continue;
    for (int b = tid; b < P.slab_bins; b += TRANSPORT_THREADS) slab[b] = 0.0;
    __syncthreads();
    TallySink S;
    S.slab = (P.slab_bins > 0) ? slab : nullptr;
    S.global_x = A.x_acc + (size_t)slot * T.n_bins;
    S.slab_lo = (long long)P.it_lo * T.G * T.mesh_n[2] * T.mesh_n[1] * T.mesh_n[0];
    S.slab_bins = P.slab_bins;
    const size_t base_in = (size_t)slot * P.cap;

    // ---- per-lane particle state (registers) ----
    bool have = false, exhausted = false;
    double x = 0, y = 0, z = 0, ux = 0, uy = 0, uz = 1, t = 0, w = 0;
    unsigned long long key = 0;
    uint32_t ctr = 0, hid = 0;
    int g = 0, cell = 0, last_surf = -1;
    uint32_t pc_coll = 0, pc_surf = 0, pc_child = 0;

    for (;;) {
      // ---------------- refill idle lanes from the slot's cursor ----------------
      unsigned need = __ballot_sync(MCDC_FULL, !have);
      if (need != 0u && !exhausted) {
        int leader = __ffs(need) - 1;
        uint32_t base = 0u;
        if (lane == leader) base = atomicAdd(A.in.cursor + slot, (uint32_t)__popc(need));
        base = __shfl_sync(MCDC_FULL, base, leader);
        if (base + (uint32_t)__popc(need) >= n_in) exhausted = true;
        if (!have) {
          uint32_t i = base + (uint32_t)__popc(need & ((1u << lane) - 1u));
          if (i < n_in) {
            size_t j = base_in + i;
            x = A.in.x[j]; y = A.in.y[j]; z = A.in.z[j]; t = A.in.t[j]; w = A.in.w[j];
            key = A.in.key[j]; hid = A.in.hid[j];
            int4 m = A.in.meta[j];
            cell = m.x;
            if (P.in_is_birth) {                         // A.6 init_child
              ctr = 0u;
              double xi_g = draw(key, ctr);
              int mat = __ldg(T.cell_mat + cell);
              g = sample_cdf(T.cdf_chi + (size_t)mat * T.G, T.G, __ldg(T.last_chi + mat), xi_g);
              double xi_mu, xi_phi;
              draw2(key, ctr, xi_mu, xi_phi);
              isotropic(xi_mu, xi_phi, ux, uy, uz);
              last_surf = -1;
            } else {
              ux = A.in.ux[j]; uy = A.in.uy[j]; uz = A.in.uz[j];
              last_surf = m.y; ctr = (uint32_t)m.z; g = m.w;
            }
            pc_coll = pc_surf = pc_child = 0u;
            have = true;
          }
        }
      }
      if (__ballot_sync(MCDC_FULL, have) == 0u) break;

      // ---------------- distances (A.2, A.4) ----------------
      double d = 0.0;
      int ev = -1, i_star = -1;
      if (have) {
        const int mat = __ldg(T.cell_mat + cell);
        const int mg = mat * T.G + g;
        const double xi = draw(key, ctr);
        const double sig_t = __ldg(T.sig_t + mg);
        const double d_coll = (sig_t > 0.0) ? -log(xi) * __ldg(T.inv_sig_t + mg) : INF;
        double d_surf = INF;
        const int e = __ldg(T.cell_off + cell + 1);
        for (int i = __ldg(T.cell_off + cell); i < e; ++i) {
          int s = __ldg(T.hs + i) >> 1;
          double u = surf_distance(T, s, s == last_surf, x, y, z, ux, uy, uz);
          if (u < d_surf) { d_surf = u; i_star = i; }
        }
        const double d_time = __ldg(T.speed + g) * (P.t_census - t);
        if (d_time <= d_surf && d_time <= d_coll) { ev = EV_CENSUS; d = d_time; }
        else if (d_surf <= d_coll)               { ev = EV_SURFACE; d = d_surf; }
        else                                     { ev = EV_COLLISION; d = d_coll; }
      }

      // ---------------- score (A.7, pre-move state), then move (A.2) ----------------
      score_track(T, S, have, x, y, z, ux, uy, uz, t, w, g, d);
      bool to_census = false;
      int n_children = 0;
      uint32_t c0 = 0u;
      if (have) {
        x += d * ux; y += d * uy; z += d * uz;
        t = (ev == EV_CENSUS) ? P.t_census : t + d * __ldg(T.inv_speed + g);
        if (ev == EV_CENSUS) {                           // A.8
          s_cnt[CNT_CENSUS][tid] += 1u;
          popw += w; popn += 1u;
          if (d > 0.0) last_surf = -1;
          if (P.is_last) s_led[LED_CENSUS_FINAL][tid] += w; else to_census = true;
          have = false;
        } else if (ev == EV_SURFACE) {                   // A.5
          pc_surf += 1u;
          const int s_star = __ldg(T.hs + i_star) >> 1;
          last_surf = s_star;
          const int bc = __ldg(T.surf_bc + s_star);
          if (bc == 1) { s_led[LED_LEAK][tid] += w; have = false; }
          else if (bc == 2) reflect(T, s_star, x, y, z, ux, uy, uz);
          else {
            int c = locate_neighbour(T, i_star, s_star, x, y, z, ux, uy, uz);
            if (c < 0) { s_led[LED_LOST][tid] += w; s_cnt[CNT_LOST][tid] += 1u; have = false; }
            else cell = c;
          }
        } else {                                         // A.6
          pc_coll += 1u;
          last_surf = -1;
          const int mat = __ldg(T.cell_mat + cell);
          const int mg = mat * T.G + g;
          const double yv = draw(key, ctr) * __ldg(T.sig_t + mg);
          const double s_tot = __ldg(T.sig_s_tot + mg);
          if (yv < s_tot) {
            double xi_g = draw(key, ctr);
            g = sample_cdf(T.cdf_s + (size_t)mg * T.G, T.G, __ldg(T.last_s + mg), xi_g * s_tot);
            double xi_mu, xi_phi;
            draw2(key, ctr, xi_mu, xi_phi);
            isotropic(xi_mu, xi_phi, ux, uy, uz);
          } else if (yv < __ldg(T.sig_sc + mg) || __ldg(T.sig_f + mg) == 0.0) {
            s_led[LED_CAPTURE][tid] += w; have = false;
          } else {
            double xi_nu = draw(key, ctr);
            n_children = (int)floor(__ldg(T.nu + mg) + xi_nu);
            c0 = ctr;
            s_led[LED_FISSION_ABS][tid] += w;
            s_led[LED_PRODUCTION][tid] += (double)n_children * w;
            pc_child += (uint32_t)n_children;
            have = false;
          }
        }
      }

      // ---------------- hand-off: census bank (A.8) ----------------
      {
        uint32_t i = warp_append(A.census_out.count + slot, to_census);
        if (to_census) {
          if (i >= P.cap) atomicExch(&A.cnt->overflow, 1);
          else {
            size_t j = (size_t)slot * P.cap + i;
            Bank &O = A.census_out;
            O.x[j] = x; O.y[j] = y; O.z[j] = z; O.ux[j] = ux; O.uy[j] = uy; O.uz[j] = uz;
            O.t[j] = t; O.w[j] = w; O.key[j] = key; O.hid[j] = hid;
            O.meta[j] = make_int4(cell, last_surf, (int)ctr, g);
          }
        }
      }
      // ---------------- hand-off: fission bank (A.6) ----------------
      {
        unsigned fis = __ballot_sync(MCDC_FULL, n_children > 0);
        if (fis != 0u) {
          int pre = n_children;                          // inclusive scan over the warp
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            int v = __shfl_up_sync(MCDC_FULL, pre, o);
            if (lane >= o) pre += v;
          }
          int total = __shfl_sync(MCDC_FULL, pre, 31);
          uint32_t base = 0u;
          if (lane == 0) base = atomicAdd(A.sec_out.count + slot, (uint32_t)total);
          base = __shfl_sync(MCDC_FULL, base, 0) + (uint32_t)(pre - n_children);
          for (int c = 0; c < n_children; ++c) {
            uint32_t i = base + (uint32_t)c;
            if (i >= P.cap) { atomicExch(&A.cnt->overflow, 1); break; }
            size_t j = (size_t)slot * P.cap + i;
            Bank &O = A.sec_out;
            O.x[j] = x; O.y[j] = y; O.z[j] = z; O.t[j] = t; O.w[j] = w; O.hid[j] = hid;
            O.key[j] = child_key(key, c0, (uint32_t)c);
            O.meta[j] = make_int4(cell, -1, 0, 0);
          }
        }
      }
      // ---------------- per-particle counters at the end of a particle's stay ----------------
      if (!have && (pc_coll | pc_surf | pc_child | (uint32_t)(ev == EV_CENSUS))) {
        s_cnt[CNT_COLL][tid] += pc_coll; s_cnt[CNT_SURF][tid] += pc_surf; s_cnt[CNT_CHILDREN][tid] += pc_child;
        if (P.record_events && A.ev != nullptr) {
          uint32_t *e4 = A.ev + (size_t)hid * 4;
          if (pc_coll) atomicAdd(e4 + 0, pc_coll);
          if (pc_surf) atomicAdd(e4 + 1, pc_surf);
          if (pc_child) atomicAdd(e4 + 2, pc_child);
          if (ev == EV_CENSUS) atomicAdd(e4 + 3, 1u);
        }
        pc_coll = pc_surf = pc_child = 0u;
      }
    }

    // ---- flush the slab into the slot's accumulator ----
    __syncthreads();
    for (int b = tid; b < P.slab_bins; b += TRANSPORT_THREADS) {
      double v = slab[b];
      if (v != 0.0) atomicAdd(S.global_x + S.slab_lo + b, v);
    }
    __syncthreads();
  }

  // ---- block totals -> global counters ----
  for (int e = 0; e < LED_N; ++e) block_atomic_add(&A.cnt->ledger[1 + e], s_led[e][tid], s_scratch);
  unsigned long long *us = (unsigned long long *)s_scratch;
  const unsigned long long nseg = (unsigned long long)s_cnt[CNT_COLL][tid] + s_cnt[CNT_SURF][tid] + s_cnt[CNT_CENSUS][tid];
  block_atomic_add_u64(&A.cnt->n[1], nseg, us);
  block_atomic_add_u64(&A.cnt->n[2], s_cnt[CNT_COLL][tid], us);
  block_atomic_add_u64(&A.cnt->n[3], s_cnt[CNT_SURF][tid], us);
  block_atomic_add_u64(&A.cnt->n[4], s_cnt[CNT_CENSUS][tid], us);
  block_atomic_add_u64(&A.cnt->n[5], s_cnt[CNT_CHILDREN][tid], us);
  block_atomic_add_u64(&A.cnt->n[6], s_cnt[CNT_LOST][tid], us);
  block_atomic_add(A.pop_w + P.k, popw, s_scratch);
  block_atomic_add_u64(A.pop_n + P.k, (unsigned long long)popn, us);
}

// ------------------------------------------------------------------------------------------------
// Batch close-out (A.9): sum += S_b, sumsq += S_b^2, S_b = 0 for every slot of the sub-batch.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_closeout(double *__restrict__ x_acc, int n_slots, int group_all,
                                                  unsigned long long n_bins, double *__restrict__ sum,
                                                  double *__restrict__ sumsq) {
  // group_all = 0: every slot is one statistical batch; 1: all slots are pieces of the same batch
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_bins; i += stride) {
    double s = 0.0, q = 0.0;
    bool any = false;
    for (int b = 0; b < n_slots; ++b) {
      double v = x_acc[(size_t)b * n_bins + i];
      if (v != 0.0) { s += v; q += v * v; x_acc[(size_t)b * n_bins + i] = 0.0; any = true; }
    }
    if (any) { sum[i] += s; sumsq[i] += group_all ? s * s : q; }
  }
}

}  // namespace mcdc
