// mcdc_kernels.cuh -- source, transport and close-out kernels (sm_100a).
//
// Scheduler (replaces the paper's Harmonize runtime): one persistent grid per census
// step.  A block adopts one statistical-batch slot at a time; its warps refill idle lanes from the
// slot's bank cursor with a ballot-aggregated atomic, keep the particle state in registers from
// segment to segment, and hand finished particles to the census bank / fission bank with
// ballot-aggregated appends.  Track-length scores go to a shared-memory copy of the step's tally slab
// (match_any-aggregated when few bins are hit) and are flushed with fp64 RED to the slot's accumulator.
#pragma once
#include "mcdc_step.cuh"

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
  double *global_x;  // this lane's slot accumulator x[slot][n_bins]
  long long slab_lo; // first global bin held by the slab
  int slab_bins;
  int aggregate;     // global mode: merge equal addresses inside the warp before the RED
};

// warp-converged sum of `val` over the lanes whose key equals the leader's, for up to `max_leaders` distinct keys;
// returns true when the caller's contribution was absorbed by a leader (leader lanes get the total in val).
template <class K>
__device__ __forceinline__ bool warp_merge_equal(K key, bool valid, double &val, int max_leaders) {
  unsigned peers = __match_any_sync(MCDC_FULL, key);
  const int my_leader = __ffs(peers) - 1;
  unsigned leaders = __ballot_sync(MCDC_FULL, valid && lane_id() == my_leader);
  if (__popc(leaders) > max_leaders) return false;          // many distinct keys: little to gain
  double mine = val;
  bool absorbed = valid && lane_id() != my_leader;
  while (leaders) {
    const int l = __ffs(leaders) - 1;
    leaders &= leaders - 1u;
    const K lk = __shfl_sync(MCDC_FULL, key, l);
    const double v = warp_sum((valid && key == lk) ? mine : 0.0);
    if (lane_id() == l) val = v;
  }
  return absorbed;
}

__device__ __forceinline__ void tally_add_converged(const TallySink &S, long long bin, double val) {
  if (S.slab == nullptr && !S.aggregate) {               // plain case (kernel-uniform): one reduction per lane, no vote
    if (bin >= 0) red_add_f64(S.global_x + bin, val);
    return;
  }
  unsigned valid = __ballot_sync(MCDC_FULL, bin >= 0);
  if (valid == 0u) return;
  if (S.slab != nullptr) {
    long long rel = bin - S.slab_lo;
    if (bin >= 0 && (rel < 0 || rel >= S.slab_bins)) {     // outside the step's slab (rounding-length pieces)
      red_add_f64(S.global_x + bin, val);
      bin = -1;
    }
    const int b = (bin >= 0) ? (int)rel : -1;
    const bool absorbed = warp_merge_equal<int>(b, b >= 0, val, 3);
    if (b >= 0 && !absorbed) atomicAdd(S.slab + b, val);
  } else if (S.aggregate) {
    double *addr = (bin >= 0) ? S.global_x + bin : nullptr;
    const bool absorbed = warp_merge_equal<unsigned long long>((unsigned long long)addr, bin >= 0, val, 3);
    if (bin >= 0 && !absorbed) red_add_f64(addr, val);
  } else if (bin >= 0) {
    red_add_f64(S.global_x + bin, val);
  }
}

// ------------------------------------------------------------------------------------------------
// A.7 track-length scoring: 4-D DDA from the pre-move state.  Warp-converged: every lane calls it,
// lanes without a segment pass active = false.
// ------------------------------------------------------------------------------------------------
template <class TBT>
__device__ __forceinline__ void score_track(const TBT &tb, const TallySink &S, bool active, double x, double y,
                                            double z, double ux, double uy, double uz, double t, double w, int g,
                                            double d) {
  const double INF = CUDART_INF;
  const Tables &T = tb.T;
  const double r[3] = {x, y, z}, o[3] = {ux, uy, uz};
  double inv_o[3];
  double u_in = 0.0, u_out = d, u_cur = 0.0;
  int idx[3] = {0, 0, 0};
  int it = 0;
  double v = 0.0;
  bool more = active;
  if (more) {
    v = tb.speed(g);
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
    u_in = fmax(u_in, (tb.time_edge(0) - t) * v);
    u_out = fmin(u_out, (tb.time_edge(T.Nt) - t) * v);
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
    const double t_in = t + u_in * tb.inv_speed(g);
    // largest it with T[it] <= t_in (binary search over the edge array)
    int lo = 0, hi = T.Nt - 1;
    while (lo < hi) {
      int mid = (lo + hi + 1) >> 1;
      if (tb.time_edge(mid) <= t_in) lo = mid; else hi = mid - 1;
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
      const double cross_t = (tb.time_edge(it + 1) - t) * v;
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
// A.7 when the mesh covers the whole geometry and the time grid covers [t0, C_K] (Tables::score_fast): the
// segment needs no clipping (u_in = 0, u_out = d), axes with a single bin never produce a crossing, and the
// time-bin index is carried by the particle (`it`, validated against the edge array, D16).  Same DDA otherwise.
// Warp-converged: every lane calls it, lanes without a segment pass active = false.
// ------------------------------------------------------------------------------------------------
template <class TBT>
__device__ __forceinline__ void score_track_fast(const TBT &tb, const TallySink &S, bool active, const PState &p, int &it_hint,
                                                 double d) {
  const double INF = CUDART_INF;
  const Tables &T = tb.T;
  const bool bx = T.mesh_n[0] > 1, by = T.mesh_n[1] > 1, bz = T.mesh_n[2] > 1;   // kernel-uniform
  int ix = 0, iy = 0, iz = 0, it = 0;
  double v = 0.0, u_cur = 0.0;
  bool more = active && d > 0.0;
  if (more) {
    v = tb.speed(p.g);
    if (bx) { const double q = floor((p.x - T.mesh_lo[0]) * T.mesh_inv_d[0]); ix = (q < 0.0) ? 0 : ((q > (double)(T.mesh_n[0] - 1)) ? T.mesh_n[0] - 1 : (int)q); }
    if (by) { const double q = floor((p.y - T.mesh_lo[1]) * T.mesh_inv_d[1]); iy = (q < 0.0) ? 0 : ((q > (double)(T.mesh_n[1] - 1)) ? T.mesh_n[1] - 1 : (int)q); }
    if (bz) { const double q = floor((p.z - T.mesh_lo[2]) * T.mesh_inv_d[2]); iz = (q < 0.0) ? 0 : ((q > (double)(T.mesh_n[2] - 1)) ? T.mesh_n[2] - 1 : (int)q); }
    // largest it with T[it] <= t: try the carried index and its successor, else search
    it = it_hint;
    double t_lo = tb.time_edge(it), t_hi = tb.time_edge(it + 1);
    if (p.t >= t_hi && it + 1 < T.Nt) { it += 1; t_lo = t_hi; t_hi = tb.time_edge(it + 1); }
    if (!(t_lo <= p.t && (p.t < t_hi || it == T.Nt - 1))) {
      int lo = 0, hi = T.Nt - 1;
      while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (tb.time_edge(mid) <= p.t) lo = mid; else hi = mid - 1;
      }
      it = lo;
    }
  }
  while (__any_sync(MCDC_FULL, more)) {
    long long bin = -1;
    double val = 0.0;
    if (more) {
      double cx = INF, cy = INF, cz = INF;
      if (bx) cx = (T.mesh_lo[0] + (double)(ix + (p.ux > 0.0 ? 1 : 0)) * T.mesh_d[0] - p.x) * p.ix;
      if (by) cy = (T.mesh_lo[1] + (double)(iy + (p.uy > 0.0 ? 1 : 0)) * T.mesh_d[1] - p.y) * p.iy;
      if (bz) cz = (T.mesh_lo[2] + (double)(iz + (p.uz > 0.0 ? 1 : 0)) * T.mesh_d[2] - p.z) * p.iz;
      if (p.ux == 0.0) cx = INF;                          // direction component 0: no crossing on that axis
      if (p.uy == 0.0) cy = INF;
      if (p.uz == 0.0) cz = INF;
      const double ct = (tb.time_edge(it + 1) - p.t) * v;
      const double u_next = fmin(fmin(d, ct), fmin(cx, fmin(cy, cz)));
      bin = ((((long long)it * T.G + p.g) * T.mesh_n[2] + iz) * T.mesh_n[1] + iy) * T.mesh_n[0] + ix;
      val = p.w * fmax(u_next - u_cur, 0.0);
      u_cur = u_next;
      if (u_next >= d) more = false;
      else {
        if (cx <= u_next) { ix += (p.ux > 0.0) ? 1 : -1; if (ix < 0 || ix >= T.mesh_n[0]) more = false; }
        if (cy <= u_next) { iy += (p.uy > 0.0) ? 1 : -1; if (iy < 0 || iy >= T.mesh_n[1]) more = false; }
        if (cz <= u_next) { iz += (p.uz > 0.0) ? 1 : -1; if (iz < 0 || iz >= T.mesh_n[2]) more = false; }
        if (ct <= u_next) { it += 1; if (it >= T.Nt) { more = false; it = T.Nt - 1; } }
      }
    }
    tally_add_converged(S, bin, val);
  }
  if (active) it_hint = it;
}

// ------------------------------------------------------------------------------------------------
// Appendix I: loc2index of a collision site for the collision-estimator tally (the paper's Fig. 3): spatial index
// floor((r - lo) / Delta) inside [lo, hi), largest it with T[it] <= t inside [T[0], T[Nt]); -1 = scores nothing.
// ------------------------------------------------------------------------------------------------
template <class TBT>
__device__ __forceinline__ long long collision_bin(const TBT &tb, double x, double y, double z, double t, int g) {
  const Tables &T = tb.T;
  const double r[3] = {x, y, z};
  int idx[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    if (!(T.mesh_lo[a] <= r[a] && r[a] < T.mesh_hi[a])) return -1;
    const int n = T.mesh_n[a];
    idx[a] = 0;
    if (n > 1) {
      const double q = floor((r[a] - T.mesh_lo[a]) / T.mesh_d[a]);
      idx[a] = (q > (double)(n - 1)) ? n - 1 : (int)q;
    }
  }
  if (!(tb.time_edge(0) <= t && t < tb.time_edge(T.Nt))) return -1;
  int lo = 0, hi = T.Nt - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (tb.time_edge(mid) <= t) lo = mid; else hi = mid - 1;
  }
  return ((((long long)lo * T.G + g) * T.mesh_n[2] + idx[2]) * T.mesh_n[1] + idx[1]) * T.mesh_n[0] + idx[0];
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
// per-thread accumulators in shared memory (no atomics: one column per thread), flushed once per block
// ------------------------------------------------------------------------------------------------
template <int NT>
struct BlockAccumT {
  double led[LED_N][NT];
  uint32_t cnt[CNT_N][NT];
  double scratch[32];
};
typedef BlockAccumT<TRANSPORT_THREADS> BlockAccum;

template <class BA>
__device__ __forceinline__ void accum_zero(BA &B) {
#pragma unroll
  for (int e = 0; e < LED_N; ++e) B.led[e][threadIdx.x] = 0.0;
#pragma unroll
  for (int e = 0; e < CNT_N; ++e) B.cnt[e][threadIdx.x] = 0u;
}

template <class BA>
__device__ __forceinline__ void accum_flush(BA &B, DevCounters *cnt) {
  const int tid = threadIdx.x;
  for (int e = 0; e < LED_N; ++e) block_atomic_add(&cnt->ledger[1 + e], B.led[e][tid], B.scratch);
  unsigned long long *us = (unsigned long long *)B.scratch;
  const unsigned long long nseg = (unsigned long long)B.cnt[CNT_COLL][tid] + B.cnt[CNT_SURF][tid] + B.cnt[CNT_CENSUS][tid];
  block_atomic_add_u64(&cnt->n[1], nseg, us);
  block_atomic_add_u64(&cnt->n[2], B.cnt[CNT_COLL][tid], us);
  block_atomic_add_u64(&cnt->n[3], B.cnt[CNT_SURF][tid], us);
  block_atomic_add_u64(&cnt->n[4], B.cnt[CNT_CENSUS][tid], us);
  block_atomic_add_u64(&cnt->n[5], B.cnt[CNT_CHILDREN][tid], us);
  block_atomic_add_u64(&cnt->n[6], B.cnt[CNT_LOST][tid], us);
}

// per-history event counts of a particle whose stay in this thread ends
template <class BA>
__device__ __forceinline__ void record_particle(BA &B, uint32_t *ev, uint32_t hid, uint32_t &pc_coll,
                                                uint32_t &pc_surf, uint32_t &pc_child, uint32_t pc_census) {
  const int tid = threadIdx.x;
  B.cnt[CNT_COLL][tid] += pc_coll; B.cnt[CNT_SURF][tid] += pc_surf; B.cnt[CNT_CHILDREN][tid] += pc_child;
  B.cnt[CNT_CENSUS][tid] += pc_census;
  if (ev != nullptr) {
    uint32_t *e4 = ev + (size_t)hid * 4;
    if (pc_coll) atomicAdd(e4 + 0, pc_coll);
    if (pc_surf) atomicAdd(e4 + 1, pc_surf);
    if (pc_child) atomicAdd(e4 + 2, pc_child);
    if (pc_census) atomicAdd(e4 + 3, pc_census);
  }
  pc_coll = pc_surf = pc_child = 0u;
}

// ------------------------------------------------------------------------------------------------
// Source kernel of the census-stepped scheduler (A.3): one thread per history of the sub-batch; histories
// whose birth time falls in census step k are appended to the live bank of their batch slot.
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

#ifndef MCDC_WARP_VARIANT   // defined once, in the host translation unit
__global__ void __launch_bounds__(256) k_source(Tables T, SourceParams P, Bank out, DevCounters *cnt) {
  __shared__ double scratch[32];
  const TB<false> tb(T);
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  bool live = i < P.n_hist;
  PState p;
  p.x = p.y = p.z = p.ux = p.uy = p.t = 0.0; p.uz = 1.0; p.w = 1.0;
  p.key = 0; p.ctr = 0; p.hid = i; p.g = 0; p.cell = -1; p.last_surf = -1;
  if (live) {
    source_position(T, P.seed_mixed, P.first_history + i, p);
    if (!P.single_step && census_index(tb, p.t) != P.k) live = false;
  }
  bool ok = false;
  if (live) ok = flight_init(tb, p, FI_SOURCE);
  const bool lost = live && !ok;
  const bool keep = live && ok;
  const int slot = keep ? (int)(i / P.hb) : -1;
  uint32_t idx = warp_append_by_slot(out.count, slot);
  if (keep) {
    if (idx >= P.cap) {
      atomicExch(&cnt->overflow, 1);
    } else {
      size_t j = (size_t)slot * P.cap + idx;
      out.x[j] = p.x; out.y[j] = p.y; out.z[j] = p.z;
      out.ux[j] = p.ux; out.uy[j] = p.uy; out.uz[j] = p.uz;
      out.t[j] = p.t; out.w[j] = p.w;
      out.key[j] = p.key;
      out.meta[j] = make_int4(p.cell, -1, (int)p.ctr, p.g);
      out.hid[j] = i;
    }
  }
  block_atomic_add(&cnt->ledger[0], live ? 1.0 : 0.0, scratch);
  block_atomic_add(&cnt->ledger[6], lost ? 1.0 : 0.0, scratch);
  block_atomic_add_u64(&cnt->n[0], live ? 1ull : 0ull, (unsigned long long *)scratch);
  block_atomic_add_u64(&cnt->n[6], lost ? 1ull : 0ull, (unsigned long long *)scratch);
}
#endif

// ------------------------------------------------------------------------------------------------
// Census-stepped transport kernel: one census step (or one fission generation inside it) for every slot.
// Particles that reach the census time are parked in the census bank (A.8); fission children go to the
// fission bank and are transported by the next launch of the same step.  Dynamic shared memory = the
// step's tally slab (tables are read from the global blob here).
// ------------------------------------------------------------------------------------------------
struct TransportArgs {
  Bank in, census_out, sec_out;
  double *x_acc;                 // [n_slots][n_bins] batch accumulators
  double *xc_acc;                // the same for the collision-estimator tally (Appendix I), nullptr = off
  DevCounters *cnt;
  double *pop_w;                 // [K]
  unsigned long long *pop_n;     // [K]
  uint32_t *ev;                  // [n_hist][4] per-history event counts of this sub-batch, or nullptr
};

#ifndef MCDC_WARP_VARIANT   // defined once, in the host translation unit
__global__ void __launch_bounds__(TRANSPORT_THREADS) k_transport(Tables T, StepParams P, TransportArgs A) {
  double *slab = reinterpret_cast<double *>(g_smem);     // [P.slab_bins]
  __shared__ BlockAccum acc;
  __shared__ int s_flag;
  const TB<false> tb(T);
  const int tid = threadIdx.x, lane = tid & 31;
  accum_zero(acc);
  double popw = 0.0;
  uint32_t popn = 0u;
  uint32_t *ev_out = P.record_events ? A.ev : nullptr;

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
    S.aggregate = 0;
    const size_t base_in = (size_t)slot * P.cap;

    bool have = false, exhausted = false;
    int fi = FI_NONE;
    PState p;
    p.x = p.y = p.z = p.ux = p.uy = p.t = p.w = 0.0; p.uz = 1.0;
    p.key = 0; p.ctr = 0; p.hid = 0; p.g = 0; p.cell = 0; p.last_surf = -1;
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
            p.x = A.in.x[j]; p.y = A.in.y[j]; p.z = A.in.z[j]; p.t = A.in.t[j]; p.w = A.in.w[j];
            p.key = A.in.key[j]; p.hid = A.in.hid[j];
            int4 m = A.in.meta[j];
            p.cell = m.x;
            if (P.in_is_birth) { p.ctr = 0u; fi = FI_CHILD; }
            else {
              p.ux = A.in.ux[j]; p.uy = A.in.uy[j]; p.uz = A.in.uz[j];
              p.last_surf = m.y; p.ctr = (uint32_t)m.z; p.g = m.w;
              fi = FI_NONE;
            }
            pc_coll = pc_surf = pc_child = 0u;
            have = true;
          }
        }
      }
      if (__ballot_sync(MCDC_FULL, have) == 0u) break;
      if (have && fi != FI_NONE) { flight_init(tb, p, fi); fi = FI_NONE; }

      double d = 0.0;
      int ev = -1, i_star = -1;
      if (have) ev = find_event(tb, p, P.t_census, d, i_star);
      score_track(tb, S, have, p.x, p.y, p.z, p.ux, p.uy, p.uz, p.t, p.w, p.g, d);
      bool to_census = false;
      int n_children = 0;
      uint32_t c0 = 0u, pc_census = 0u;
      if (have) {
        p.x += d * p.ux; p.y += d * p.uy; p.z += d * p.uz;
        p.t = (ev == EV_CENSUS) ? P.t_census : p.t + d * tb.inv_speed(p.g);
        if (ev == EV_CENSUS) {                           // A.8
          pc_census = 1u;
          popw += p.w; popn += 1u;
          if (d > 0.0) p.last_surf = -1;
          if (P.is_last) acc.led[LED_CENSUS_FINAL][tid] += p.w; else to_census = true;
          have = false;
        } else if (ev == EV_SURFACE) {
          pc_surf += 1u;
          have = surface_event(tb, p, i_star, &acc.led[LED_LEAK][tid], &acc.led[LED_LOST][tid], &acc.cnt[CNT_LOST][tid]);
        } else {
          pc_coll += 1u;
          if (A.xc_acc != nullptr) {                     // Appendix I, with the weight the particle arrives with
            const long long cb = collision_bin(tb, p.x, p.y, p.z, p.t, p.g);
            if (cb >= 0) atomicAdd(A.xc_acc + (size_t)slot * T.n_bins + cb, p.w / tb.sig_t(tb.cell_mat(p.cell) * T.G + p.g));
          }
          int r = collision_event(tb, p, c0, &acc.led[LED_CAPTURE][tid], &acc.led[LED_FISSION_ABS][tid],
                                  &acc.led[LED_PRODUCTION][tid], &acc.led[LED_VR_GAIN][tid], &acc.led[LED_VR_LOSS][tid]);
          if (r == -1) fi = FI_SCATTER; else have = false;
          if (r > 0) { n_children = r; pc_child += (uint32_t)r; }
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
            O.x[j] = p.x; O.y[j] = p.y; O.z[j] = p.z; O.ux[j] = p.ux; O.uy[j] = p.uy; O.uz[j] = p.uz;
            O.t[j] = p.t; O.w[j] = p.w; O.key[j] = p.key; O.hid[j] = p.hid;
            O.meta[j] = make_int4(p.cell, p.last_surf, (int)p.ctr, p.g);
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
            O.x[j] = p.x; O.y[j] = p.y; O.z[j] = p.z; O.t[j] = p.t; O.w[j] = p.w; O.hid[j] = p.hid;
            O.key[j] = child_key(p.key, c0, (uint32_t)c);
            O.meta[j] = make_int4(p.cell, -1, 0, 0);
          }
        }
      }
      if (!have && ev >= 0) record_particle(acc, ev_out, p.hid, pc_coll, pc_surf, pc_child, pc_census);
    }

    // ---- flush the slab into the slot's accumulator ----
    __syncthreads();
    for (int b = tid; b < P.slab_bins; b += TRANSPORT_THREADS) {
      double v = slab[b];
      if (v != 0.0) red_add_f64(S.global_x + S.slab_lo + b, v);
    }
    __syncthreads();
  }
  accum_flush(acc, A.cnt);
  block_atomic_add(A.pop_w + P.k, popw, acc.scratch);
  block_atomic_add_u64(A.pop_n + P.k, (unsigned long long)popn, (unsigned long long *)acc.scratch);
}
#endif

// ------------------------------------------------------------------------------------------------
// Population control at census (Appendix G.3; "time-dependent population control"), census-stepped
// scheduler.  Per batch slot: k_pc_weight sums the arriving weight in 2^-40 fixed point (an integer sum: the
// result does not depend on the order of the bank), k_pc_apply turns every particle of the census bank into
// floor(w / w_t + xi) particles of weight w_t = W / target in the next live bank.  Grid: (chunks of 256, slots).
// ------------------------------------------------------------------------------------------------
#define MCDC_FIX40 1099511627776.0   // 2^40

#ifndef MCDC_WARP_VARIANT   // defined once, in the host translation unit
__global__ void __launch_bounds__(256) k_pc_weight(Bank in, uint32_t cap, unsigned long long *wfix) {
  __shared__ unsigned long long scratch[32];
  const int slot = blockIdx.y;
  const uint32_t n = min(in.count[slot], cap);
  if (blockIdx.x * blockDim.x >= n) return;              // (grids are sized for the bank capacity: no host read of the counts)
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long v = 0ull;
  if (i < n) v = (unsigned long long)(in.w[(size_t)slot * cap + i] * MCDC_FIX40);   // truncation, as the oracle's cast
  block_atomic_add_u64(wfix + slot, v, scratch);
}
#endif

struct PcParams {
  uint32_t cap;
  int k;                              // census index
  unsigned long long target;          // particles per batch after the control
  double w_out;                       // > 0: weight given to every copy (generation control, Appendix H.3); else w_t
};

#ifndef MCDC_WARP_VARIANT   // defined once, in the host translation unit
__global__ void __launch_bounds__(256) k_pc_apply(Bank in, Bank out, PcParams P, const unsigned long long *wfix,
                                                  DevCounters *cnt, double *pop_w_after, unsigned long long *pop_n_after) {
  __shared__ double scratch[32];
  const int slot = blockIdx.y, lane = lane_id();
  const uint32_t n_in = min(in.count[slot], P.cap);
  if (blockIdx.x * blockDim.x >= n_in) return;
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long W = wfix[slot];
  const bool have = i < n_in && W != 0ull;
  const size_t j = (size_t)slot * P.cap + (have ? i : 0u);
  const double w_t = ((double)W / MCDC_FIX40) / (double)P.target;
  const double w_new = (P.w_out > 0.0) ? P.w_out : w_t;
  double w = 0.0, gain = 0.0, loss = 0.0;
  unsigned long long key = 0ull;
  uint32_t ctr = 0u;
  int4 m = make_int4(0, -1, 0, 0);
  int n = 0;
  if (have) {
    w = in.w[j]; key = in.key[j]; m = in.meta[j]; ctr = (uint32_t)m.z;
  }
  const double xi = draw(key, ctr);                      // the particle's own stream
  if (have) {
    n = (int)floor(w / w_t + xi);
    const double dw = (double)n * w_t - w;
    if (dw > 0.0) gain = dw; else loss = -dw;
  }
  // ballot-free inclusive scan of the copies over the warp, one atomic per warp on the slot's counter
  int pre = n;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(MCDC_FULL, pre, o);
    if (lane >= o) pre += v;
  }
  const int total = __shfl_sync(MCDC_FULL, pre, 31);
  uint32_t base = 0u;
  if (lane == 0 && total > 0) base = atomicAdd(out.count + slot, (uint32_t)total);
  base = __shfl_sync(MCDC_FULL, base, 0) + (uint32_t)(pre - n);
  if (n > 0) {
    const double x = in.x[j], y = in.y[j], z = in.z[j], ux = in.ux[j], uy = in.uy[j], uz = in.uz[j], t = in.t[j];
    const uint32_t hid = in.hid[j];
    for (int c = 0; c < n; ++c) {
      const uint32_t o = base + (uint32_t)c;
      if (o >= P.cap) { atomicExch(&cnt->overflow, 1); break; }
      const size_t q = (size_t)slot * P.cap + o;
      out.x[q] = x; out.y[q] = y; out.z[q] = z; out.ux[q] = ux; out.uy[q] = uy; out.uz[q] = uz; out.t[q] = t;
      out.w[q] = w_new; out.hid[q] = hid;
      out.key[q] = (c == 0) ? key : child_key(key, ctr, (uint32_t)c);   // copy 0 keeps its stream
      out.meta[q] = make_int4(m.x, m.y, (c == 0) ? (int)ctr : 0, m.w);
    }
  }
  block_atomic_add(&cnt->ledger[1 + LED_VR_GAIN], gain, scratch);
  block_atomic_add(&cnt->ledger[1 + LED_VR_LOSS], loss, scratch);
  block_atomic_add_u64(&cnt->n[7], (have && n == 0) ? 1ull : 0ull, (unsigned long long *)scratch);
  block_atomic_add_u64(&cnt->n[8], (n > 1) ? (unsigned long long)(n - 1) : 0ull, (unsigned long long *)scratch);
  block_atomic_add(pop_w_after + P.k, (double)n * w_new, scratch);
  block_atomic_add_u64(pop_n_after + P.k, (unsigned long long)n, (unsigned long long *)scratch);
}
#endif

#ifndef MCDC_WARP_VARIANT   // defined once, in the host translation unit
// The same control applied IN PLACE (census-step mode of k_warp): the census bank itself becomes the next live bank.
// A record that survives keeps its place and only its weight and counter are rewritten (copy 0 keeps key and stream);
// a record that is removed (n = 0) is marked as a hole (meta.x = -1: the refill of the next launch skips it); copies
// j >= 1 are appended behind the arrivals.  n_arrived[slot] is the count of the bank BEFORE any append (a snapshot the
// host queues in front of this kernel).  Traffic per particle: 32 B read + 12 B written instead of 92 B + 92 B.
__global__ void __launch_bounds__(256) k_pc_apply_inplace(Bank bank, const uint32_t *n_arrived, PcParams P,
                                                          const unsigned long long *wfix, DevCounters *cnt,
                                                          double *pop_w_after, unsigned long long *pop_n_after) {
  const int slot = blockIdx.y, lane = lane_id();
  const uint32_t n_in = min(n_arrived[slot], P.cap);
  if (blockIdx.x * blockDim.x >= n_in) return;
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long W = wfix[slot];
  const bool have = i < n_in && W != 0ull;
  const size_t j = (size_t)slot * P.cap + (have ? i : 0u);
  const double w_t = ((double)W / MCDC_FIX40) / (double)P.target;
  const double w_new = (P.w_out > 0.0) ? P.w_out : w_t;
  double w = 0.0, gain = 0.0, loss = 0.0;
  unsigned long long key = 0ull;
  uint32_t ctr = 0u;
  int4 m = make_int4(0, -1, 0, 0);
  int n = 0;
  if (have) { w = bank.w[j]; key = bank.key[j]; m = bank.meta[j]; ctr = (uint32_t)m.z; }
  // W == 0: every arrival of this batch weighs less than 2^-40, so the fixed-point sum is zero and G.3 hands back an
  // EMPTY bank without touching a counter (k_pc_apply: out.count stays 0).  In place that means every arrival
  // becomes a hole; left alone, the next launch would pick all of them up as live particles.
  if (i < n_in && W == 0ull) bank.meta[(size_t)slot * P.cap + i].x = -1;
  const double xi = draw(key, ctr);                      // the particle's own stream
  if (have) {
    n = (int)floor(w / w_t + xi);
    const double dw = (double)n * w_t - w;
    if (dw > 0.0) gain = dw; else loss = -dw;
    if (n == 0) bank.meta[j].x = -1;                     // a hole
    else { bank.w[j] = w_new; bank.meta[j].z = (int)ctr; }
  }
  const int extra = n > 1 ? n - 1 : 0;
  int pre = extra;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(MCDC_FULL, pre, o);
    if (lane >= o) pre += v;
  }
  const int total = __shfl_sync(MCDC_FULL, pre, 31);
  uint32_t base = 0u;
  if (lane == 0 && total > 0) base = atomicAdd(bank.count + slot, (uint32_t)total);
  base = __shfl_sync(MCDC_FULL, base, 0) + (uint32_t)(pre - extra);
  if (extra > 0) {
    const double x = bank.x[j], y = bank.y[j], z = bank.z[j], ux = bank.ux[j], uy = bank.uy[j], uz = bank.uz[j], t = bank.t[j];
    const uint32_t hid = bank.hid[j];
    for (int c = 1; c <= extra; ++c) {
      const uint32_t o = base + (uint32_t)(c - 1);
      if (o >= P.cap) { atomicExch(&cnt->overflow, 1); break; }
      const size_t q = (size_t)slot * P.cap + o;
      bank.x[q] = x; bank.y[q] = y; bank.z[q] = z; bank.ux[q] = ux; bank.uy[q] = uy; bank.uz[q] = uz; bank.t[q] = t;
      bank.w[q] = w_new; bank.hid[q] = hid;
      bank.key[q] = child_key(key, ctr, (uint32_t)c);
      bank.meta[q] = make_int4(m.x, m.y, 0, m.w);
    }
  }
  // block totals: warp sums first, one barrier, six global atomics per block (six block-wide reductions with two
  // barriers each made this kernel compute-bound: 470 -> 286 us per census with the in-place rewrite, then this)
  __shared__ double s_tot[3][8];
  __shared__ unsigned long long s_cnt[3][8];
  const int wid = threadIdx.x >> 5;
  const double g_ = warp_sum(gain), l_ = warp_sum(loss), a_ = warp_sum((double)n * w_new);
  const unsigned long long r_ = (unsigned long long)__popc(__ballot_sync(MCDC_FULL, have && n == 0));
  const unsigned long long e_ = (unsigned long long)__reduce_add_sync(MCDC_FULL, (unsigned)extra);
  const unsigned long long n_ = (unsigned long long)__reduce_add_sync(MCDC_FULL, (unsigned)n);
  if (lane == 0) { s_tot[0][wid] = g_; s_tot[1][wid] = l_; s_tot[2][wid] = a_; s_cnt[0][wid] = r_; s_cnt[1][wid] = e_; s_cnt[2][wid] = n_; }
  __syncthreads();
  if (threadIdx.x < 6) {
    const int q = threadIdx.x;
    if (q < 3) {
      double t = 0.0;
      for (int k = 0; k < 8; ++k) t += s_tot[q][k];
      double *dst = q == 0 ? &cnt->ledger[1 + LED_VR_GAIN] : q == 1 ? &cnt->ledger[1 + LED_VR_LOSS] : pop_w_after + P.k;
      if (t != 0.0) atomicAdd(dst, t);
    } else {
      unsigned long long t = 0ull;
      for (int k = 0; k < 8; ++k) t += s_cnt[q - 3][k];
      unsigned long long *dst = q == 3 ? &cnt->n[7] : q == 4 ? &cnt->n[8] : pop_n_after + P.k;
      if (t != 0ull) atomicAdd(dst, t);
    }
  }
}
#endif

// ------------------------------------------------------------------------------------------------
// Global fission queue and launch arguments of the asynchronous history kernel k_warp (mcdc_warp.cuh).
// ------------------------------------------------------------------------------------------------
struct FissionQueue {             // ring buffer in HBM, structure of arrays, capacity mask+1 (power of two)
  double *x, *y, *z, *t, *w;      // w is read and written only when a technique makes weights differ from 1
  unsigned long long *key;
  int4 *meta;                     // {cell, census index k, history id (when events are recorded), batch slot}
  uint32_t *flag;                 // entry i is readable when flag[i & mask] == (uint32)(i + 1)
  uint32_t mask;
  unsigned long long *head_tail;  // [0] consumers' cursor, [1] producers' cursor (monotonic over launches)
};

struct HistoryArgs {
  FissionQueue q;
  uint32_t *hist_cursor;          // next source history of this sub-batch
  unsigned long long seed_mixed, first_history;
  uint32_t n_hist, hb;            // histories in the sub-batch, histories per slot
  uint32_t src_chunk;             // source histories a warp reserves per global atomic
  uint32_t n_slots, n_chunks;     // batch slots of the sub-batch; chunks in all = n_slots * ceil(hb / src_chunk)
  double *x_acc;
  double *xc_acc;                 // collision-estimator accumulators (Appendix I; k_warp<WEIGHTED> only), nullptr = off
  DevCounters *cnt;
  double *pop_w;
  unsigned long long *pop_n;
  uint32_t *ev;
  int aggregate;
  uint32_t smem_tables;           // bytes of dynamic shared memory in front of the census arrays
  uint32_t pool_slots;            // particles held in each warp's shared-memory pool
  uint32_t pool_reserve;          // slots a refill leaves free for the children of fissions
  // census-step mode of k_warp<WEIGHTED> (population control, Appendix G.3): one launch transports one census step.
  // Particles come from the live bank `in` (survivors of the control at the previous census) and from the source
  // histories born in this step; a particle that reaches the census time is parked in `census_out` instead of going on.
  int step_mode, step_k, step_source, step_single;   // 0 off, 1 census step, 2 generation (Appendix H); census index;
                                                     // sources may be born in this launch; all of them are
  uint32_t bank_cap;              // bank capacity per batch slot
  Bank in, census_out;
};

__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t *p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_u32(uint32_t *p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_volatile_u64(const unsigned long long *p) {
  unsigned long long v;
  asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}

// ------------------------------------------------------------------------------------------------
// Batch close-out (A.9): sum += S_b, sumsq += S_b^2, S_b = 0 for every slot of the sub-batch.
// ------------------------------------------------------------------------------------------------
#ifndef MCDC_WARP_VARIANT   // defined once, in the host translation unit
__global__ void __launch_bounds__(256) k_closeout(double *__restrict__ x_acc, int n_slots, int group_all,
                                                  unsigned long long n_bins, double *__restrict__ sum,
                                                  double *__restrict__ sumsq) {
  // group_all = 0: every slot is one statistical batch; 1: all slots are pieces of the same batch
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_bins; i += stride) {
    double s = 0.0, q = 0.0;
    bool any = false;
    int b = 0;
    for (; b + 4 <= n_slots; b += 4) {                   // four slots at a time: four independent loads in flight per thread
      double v[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) v[k] = x_acc[(size_t)(b + k) * n_bins + i];
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (v[k] != 0.0) { s += v[k]; q += v[k] * v[k]; x_acc[(size_t)(b + k) * n_bins + i] = 0.0; any = true; }
    }
    for (; b < n_slots; ++b) {
      double v = x_acc[(size_t)b * n_bins + i];
      if (v != 0.0) { s += v; q += v * v; x_acc[(size_t)b * n_bins + i] = 0.0; any = true; }
    }
    if (any) { sum[i] += s; sumsq[i] += group_all ? s * s : q; }
  }
}
#endif

// ------------------------------------------------------------------------------------------------
// A.9 read-out for large meshes: mean = sum / N, sdev = sqrt((sumsq / hb^2 / B - mean^2) / (B - 1)) per bin
// ------------------------------------------------------------------------------------------------
#ifndef MCDC_WARP_VARIANT   // defined once, in the host translation unit
__global__ void __launch_bounds__(256) k_statistics(const double *__restrict__ sum, const double *__restrict__ sumsq,
                                                    unsigned long long n_bins, double N, double B,
                                                    double *__restrict__ mean, double *__restrict__ sdev) {
  const double hb = N / B;
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_bins; i += stride) {
    const double mu = sum[i] / N;
    double sd = 0.0;
    if (B > 1.0) {
      const double m2 = sumsq[i] / (hb * hb) / B;
      const double var = (m2 - __dmul_rn(mu, mu)) / (B - 1.0);   // no FMA contraction: same bits as the host loop
      sd = var > 0.0 ? sqrt(var) : 0.0;
    }
    mean[i] = mu; sdev[i] = sd;
  }
}
#endif

}  // namespace mcdc
