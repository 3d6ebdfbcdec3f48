// mcdc_warp.cuh -- k_warp: the event-based history kernel (default scheduler, MCDC_SCHED_ASYNC).
//
// Replaces the paper's Harmonize runtime ("segregating them into like-operations ... executed
// together in batches") with an ON-CHIP, PER-WARP event scheduler.  Every warp owns a pool of W particles in shared
// memory (structure of arrays) and three index stacks -- F (needs a flight), C (collided), FREE -- that it edits
// with ballots only: no atomics, no block barriers, warps never wait for one another.  Each round the warp picks
// the stack that fills all 32 lanes and runs ONE kind of work on it:
//   R  refill   free slots take fission children from the global ring queue, then new source histories (A.3, A.6)
//   F  flight   distances, event choice, track-length score, move (A.2, A.4, A.7); census bookkeeping (A.8) and
//               the surface event (A.5) are finished in the same round -- with a certified neighbour a crossing
//               is a table look-up
//   C  collide  reaction choice, scattering or fission (A.6); a fission parent continues as its first child,
//               the other children go to the global queue
// Particle records never travel through HBM; only the fission queue, the batch accumulators (fp64 RED) and the
// counters do.  Trajectories depend on (seed, history id, lineage) alone, so the processing order is free
// (DESIGN.md section 5).  Analog transport: every weight is 1 and is not stored.
#pragma once
#include "mcdc_kernels.cuh"

namespace mcdc {

// ---- slow paths: rare, not inlined, and they read the tables from global memory (device copy of Tables) ----

// A.5 transmission without a certified neighbour: candidate cells of half-space `idx` of `cell`, then every cell
// (RGN: the problem holds general CSG regions, Appendix J -- instantiations of their own, so that the expression
// evaluator is no part of the kernels that never run it)
template <bool RGN>
static __device__ __noinline__ int slow_cross(const Tables *gT, int cell, int idx, int s_star, double x, double y, double z,
                                       double ux, double uy, double uz) {
  const TB<false> tb(*gT);
  const int slot = tb.cell_off(cell) + idx;
  return locate_neighbour<RGN>(tb, slot, s_star, x, y, z, ux, uy, uz);
}
// A.5 reflection off a surface that is not an axis-aligned plane
static __device__ __noinline__ void slow_reflect(const Tables *gT, int s, int type, double x, double y, double z, double *u) {
  const TB<false> tb(*gT);
  reflect(tb, s, type, x, y, z, u[0], u[1], u[2]);
}
// A.3 cell of a source particle
template <bool RGN>
static __device__ __noinline__ int slow_locate_source(const Tables *gT, double x, double y, double z, double ux, double uy,
                                               double uz) {
  const TB<false> tb(*gT);
  return locate_source<RGN>(tb, x, y, z, ux, uy, uz);
}
// A.4 distance to a surface that is neither an axis-aligned plane face nor a z-cylinder
static __device__ __noinline__ double slow_distance(const Tables *gT, int s, int type, bool on, double x, double y, double z,
                                             double ux, double uy, double uz) {
  const TB<false> tb(*gT);
  return surf_distance(tb, s, type, on, x, y, z, ux, uy, uz, 1.0 / ux, 1.0 / uy, 1.0 / uz);
}

// A.6 fission children that do not fit their parent's pool go to the global ring queue (SoA entries, per-entry
// sequence flags published with st.release).  Warp-converged: every lane calls it; lanes without children pass
// n_push = 0.  Out of line: it runs in under 1 % of the collision rounds and its ~470 instructions sat in the middle
// of the C phase (profiles/r01g).
static __device__ __noinline__ void slow_publish_children(FissionQueue q, DevCounters *cnt, bool weighted, double x, double y,
                                                   double z, double t, double w, unsigned long long key, uint32_t c0,
                                                   int n_push, int pre, int total, int4 qm) {
  const int lane = threadIdx.x & 31;
  unsigned long long *q_head = q.head_tail, *q_tail = q.head_tail + 1;
  const unsigned long long q_cap = (unsigned long long)q.mask + 1ull;
  unsigned long long qb = 0ull;
  int okq = 1;
  if (lane == 0) {
    // consumers advance head before they read their entries: up to one claimed-but-unread entry per thread of the
    // launch may still be in use behind head, so that many entries stay out of the producers' reach
    qb = atomicAdd(q_tail, (unsigned long long)total);
    if (qb + (unsigned long long)total - ld_volatile_u64(q_head) + (unsigned long long)gridDim.x * blockDim.x > q_cap) okq = 0;
  }
  qb = __shfl_sync(MCDC_FULL, qb, 0) + (unsigned long long)(pre - n_push);
  okq = __shfl_sync(MCDC_FULL, okq, 0);
  if (!okq && lane == 0) atomicExch(&cnt->overflow, 1);
  if (n_push > 0 && okq) {
    for (int c = 0; c < n_push; ++c) {
      const uint32_t j = (uint32_t)(qb + (unsigned long long)c) & q.mask;
      q.x[j] = x; q.y[j] = y; q.z[j] = z; q.t[j] = t;
      if (weighted) q.w[j] = w;
      q.key[j] = child_key(key, c0, (uint32_t)(c + 1));
      q.meta[j] = qm;
    }
    __threadfence();
    for (int c = 0; c < n_push; ++c) {
      const unsigned long long qi = qb + (unsigned long long)c;
      st_release_u32(q.flag + ((uint32_t)qi & q.mask), (uint32_t)(qi + 1ull));
    }
  }
}

// Appendix I: one collision-estimator score (only runs that enabled the tally come here)
static __device__ __noinline__ void slow_score_collision(const Tables *gT, double *xc_slot, double x, double y, double z, double t,
                                                  int g, double w, int mg) {
  const TB<false> tb(*gT);
  const long long cb = collision_bin(tb, x, y, z, t, g);
  if (cb >= 0) red_add_f64(xc_slot + cb, w / tb.sig_t(mg));
}

// A.7 for segments that may touch several tally bins (4-D DDA).  Warp-converged: every lane calls it.
template <bool STAGED>
__device__ __forceinline__ void general_score(const Tables &Tg, double *x_acc_slot, int aggregate, bool active,
                                           const double *pool, uint32_t N, uint32_t gi, int g, int pk, double d, double w) {
  // the pre-move state is still in the pool: five pairs (x y)(z t)(ux uy)(uz 1/ux)(1/uy 1/uz) per slot
  (void)N;
  const double2 *pp = reinterpret_cast<const double2 *>(pool) + 5u * gi;
  const double2 xy = pp[0], zt = pp[1], u01 = pp[2], u2i0 = pp[3], i12 = pp[4];
  const double x = xy.x, y = xy.y, z = zt.x, t = zt.y, ux = u01.x, uy = u01.y, uz = u2i0.x, ix = u2i0.y, iy = i12.x, iz = i12.y;
  // Tg is the kernel's parameter block (constant bank) when this is inlined -- reading the mesh constants through the
  // device-memory copy of the tables made every DDA step wait on global loads (config 2: long_scoreboard 3.2 per issue)
  const TB<STAGED> tb(Tg);
  TallySink S;
  S.slab = nullptr; S.global_x = x_acc_slot; S.slab_lo = 0; S.slab_bins = 0; S.aggregate = aggregate;
  if (Tg.score_fast) {
    PState p;
    p.x = x; p.y = y; p.z = z; p.ux = ux; p.uy = uy; p.uz = uz; p.ix = ix; p.iy = iy; p.iz = iz; p.t = t; p.w = w;
    p.key = 0ull; p.ctr = 0u; p.hid = 0u; p.g = g; p.cell = 0; p.last_surf = -1;
    int it = tb.template ld<int>(Tg.o_it0_k, pk);
    score_track_fast(tb, S, active, p, it, d);
  } else {
    score_track(tb, S, active, x, y, z, ux, uy, uz, t, w, g, d);
  }
}

// 0 < v < +inf, decided on the bit pattern (two integer instructions instead of two fp64 compares)
__device__ __forceinline__ bool pos_finite(double v) {
  return (unsigned long long)(__double_as_longlong(v) - 1ll) < 0x7FEFFFFFFFFFFFFFull;
}

__device__ __forceinline__ uint32_t lanes_below(unsigned m, int lane) { return (uint32_t)__popc(m & ((1u << lane) - 1u)); }

// bytes of shared memory per pool slot: the flight record x y z t ux uy uz 1/ux 1/uy 1/uz (10 x f64, contiguous), the key and
// the unused half of the last Philox block (2 x u64), ctr, cell | last, meta [, history id] (u32 each), 3 stack entries
// (+ the weight, one more f64, when a technique of Appendix G makes weights differ from 1)
__host__ __device__ inline size_t warp_pool_bytes_per_slot(bool record, bool weighted) {
  return 80 + 16 + 12 + 3 + (record ? 4 : 0) + (weighted ? 8 : 0);
}

// Copies of the census-weight array of a block (weighted variants): lane l adds to copy l & 3.  Adds of several lanes to ONE
// shared-memory double serialise in a compare-and-swap loop (12 % of the weighted kernel's samples, profiles/r02k); four
// copies spread the lanes of a round that reach the same census.
#define POPW_COPIES 4
// ... of which the census-step and generation variants (VARIANT >= 2) need only one: they sum the census weight in a
// register per lane and add once per warp to copy 0.  With K near 4095 three unused copies cost 96 KB of the pool.
__host__ __device__ constexpr int popw_copies(int variant) { return variant >= 2 ? 1 : POPW_COPIES; }

struct WarpShared {                // block-wide totals (static shared memory)
  double led[LED_N];
  unsigned long long n_coll, n_seg, n_census, n_children, n_lost, n_src;
  double wled[32][LED_N];            // weighted runs: per-warp ledger sums (lane 0 of the warp adds without atomics; leaks: the warp's lanes)
  uint32_t n_leak;                   // analog runs: particles that leaked from this block (unit weights: a native 32-bit add)
  uint32_t wcnt[32][8];              // per-warp event counts (only lane 0 of the warp touches its row)
};

// VARIANT: 0 analog (unit weights, not stored); 1 weighted (Appendix G.1 / G.2, collision tally); 2 weighted, census-step
// mode (G.3); 3 weighted, generation mode (H).  Separate instantiations: every variant carries only its own code --
// the kernel is sensitive to its instruction-cache footprint (profiles/r01e, r01f).
// ONEBIN: every cell lies in one spatial tally bin and every census interval in one time bin (Tables::all_one_bin, found
// at create): every score is a single RED and the 4-D DDA scorer is not compiled in.  It is ~1000 instructions that
// such problems never execute, in the middle of the flight phase: leaving it out is worth 8 % on config 3 (r01f).
// SCORE: 0 = general (DDA scorer compiled in, one-bin shortcut and in-warp merge chosen at run time); 1 = ONEBIN, one RED
// per score; 2 = ONEBIN on a tiny mesh, equal addresses merged inside the warp before the RED.
// RGN: cells may be general CSG regions (Appendix J).  A region cell has no faces and no certified neighbours: every one of
// its surfaces is an "other" entry, every crossing takes the search of A.5 with the expression evaluator (slow_cross<true>),
// and source particles are located with it; everything else of the kernel is unchanged.  Always with SCORE = 0.
#ifdef MCDC_WARP_MAXNREG
#define MCDC_WARP_BOUNDS __maxnreg__(MCDC_WARP_MAXNREG)
#else
#define MCDC_WARP_BOUNDS __launch_bounds__(NT, 1)
#endif
template <bool STAGED, bool RECORD, int VARIANT, int SCORE, int NT, bool RGN = false>
__global__ void MCDC_WARP_BOUNDS k_warp(Tables T, HistoryArgs A) {
  constexpr bool ONEBIN = SCORE != 0;
  constexpr bool WEIGHTED = VARIANT != 0;
  constexpr int NW = NT / 32;
  const double INF = CUDART_INF;
  __shared__ WarpShared sh;
  const TB<STAGED> tb(T);
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const uint32_t W = A.pool_slots;                    // slots per warp
  const uint32_t N = W * (uint32_t)NW;
  // ---- carve the dynamic shared memory: [staged tables][census populations][pool arrays][stacks] ----
  // Offsets from pool_off (N = slots of the block):
  //   flight records, 80 bytes per slot: (x y)(z t)(ux uy)(uz 1/ux)(1/uy 1/uz) as five 16-byte pairs -> PP(pair, slot), one
  //     LDS.128 each at a constant offset from the slot's address (one multiply per round instead of one per array; 5
  //     pairs per slot keep a 32-slot gather spread over the bank groups as the slot index itself: 5 is odd);
  //     single fields -> PD(k, slot), k = D_X .. D_IZ
  //   N * 80:  (key, half block) per slot -> PKC / PK / PC; half block = second half of Philox block ctr >> 1, valid while
  //     ctr is odd (Appendix B: "may cache the half-block")
  //   N * 96:  [weight, f64 per slot -> PW(slot)]   (WEIGHTED)
  //   then u32 arrays ctr, cell | last << 16, meta = g | census index << 8 | batch slot << 20, [history id] -> PU(k, slot)
  //     (4-byte stride: the counter store of every flight round stays free of bank conflicts)
  //   then the u8 stacks F, C, FREE -> PL(k, position)
  uint32_t *s_popn = reinterpret_cast<uint32_t *>(g_smem + A.smem_tables);
  double *s_popw = reinterpret_cast<double *>(g_smem + A.smem_tables + (uint32_t)(((size_t)T.K * 4 + 15) / 16 * 16));   // WEIGHTED only
  const uint32_t pool_off = A.smem_tables + (uint32_t)(((size_t)T.K * 4 + 15) / 16 * 16) +
                            (WEIGHTED ? (uint32_t)(((size_t)T.K * 8 * popw_copies(VARIANT) + 15) / 16 * 16) : 0u);
#define PP(pr, slot) (*reinterpret_cast<double2 *>(g_smem + pool_off + (slot) * 80u + (uint32_t)(pr) * 16u))
#define PD(k, slot) (*reinterpret_cast<double *>(g_smem + pool_off + (slot) * 80u + (uint32_t)(k) * 8u))
#define PK(slot) (*reinterpret_cast<unsigned long long *>(g_smem + pool_off + N * 80u + (slot) * 16u))
#define PC(slot) (*reinterpret_cast<unsigned long long *>(g_smem + pool_off + N * 80u + (slot) * 16u + 8u))
#define PKC(slot) (*reinterpret_cast<ulonglong2 *>(g_smem + pool_off + N * 80u + (slot) * 16u))
#define PW(slot) (*reinterpret_cast<double *>(g_smem + pool_off + N * 96u + (slot) * 8u))
#define PU(k, slot) (*reinterpret_cast<uint32_t *>(g_smem + pool_off + N * (WEIGHTED ? 104u : 96u) + ((uint32_t)(k) * N + (slot)) * 4u))
#define PL(k, pos) (*reinterpret_cast<uint8_t *>(g_smem + pool_off + ((WEIGHTED ? 104u : 96u) + (RECORD ? 16u : 12u)) * N + (uint32_t)(k) * N + (pos)))
  enum { D_X = 0, D_Y, D_Z, D_T, D_UX, D_UY, D_UZ, D_IX, D_IY, D_IZ, P_XY = 0, P_ZT, P_U01, P_U2I0, P_I12,
         U_CTR = 0, U_CL, U_META, U_HID, L_F = 0, L_C, L_FREE };

  if (STAGED) {
    const uint4 *src = reinterpret_cast<const uint4 *>(T.blob);
    uint4 *dst = reinterpret_cast<uint4 *>(g_smem);
    for (uint32_t i = tid; i < T.hot_bytes / 16u; i += NT) dst[i] = src[i];
  }
  for (int k = tid; k < T.K; k += NT) s_popn[k] = 0u;
  if (WEIGHTED) for (int k = tid; k < T.K * popw_copies(VARIANT); k += NT) s_popw[k] = 0.0;
  if (tid == 0) {
    for (int e = 0; e < LED_N; ++e) sh.led[e] = 0.0;
    sh.n_coll = sh.n_seg = sh.n_census = sh.n_children = sh.n_lost = sh.n_src = 0ull; sh.n_leak = 0u;
  }
  if (lane < 8) sh.wcnt[wid][lane] = 0u;
  if (lane < LED_N) sh.wled[wid][lane] = 0.0;
  const uint32_t lb = (uint32_t)wid * W;               // first slot of this warp
  for (uint32_t i = lane; i < W; i += 32) PL(L_FREE, lb + i) = (uint8_t)(W - 1u - i);
  __syncthreads();

  unsigned long long *q_head = A.q.head_tail, *q_tail = A.q.head_tail + 1;
  const Tables *gT = T.self_dev;
  const int G = T.G;
  const long long n_spatial = (long long)T.mesh_n[0] * T.mesh_n[1] * T.mesh_n[2];
  // indices into all the batch accumulators fit 32 bits: no 64-bit multiplies per score
  const bool bins32 = T.n_bins * (unsigned long long)max(A.n_slots, 1u) < 0x7FFFFFFFull;
  // warp-uniform scheduler state
  uint32_t nF = 0u, nC = 0u, nFree = W, dry = 0u, r_calls = 0u;
  uint32_t src_next = 0u, src_end = 0u;                // the warp's chunk of source histories
  bool src_exhausted = false;
  constexpr bool step_mode = VARIANT >= 2;             // census-step mode (Appendix G.3) or generation mode (H)
  constexpr bool gen_mode = VARIANT == 3;              // k-eigenvalue: `in` holds birth records, children go to `census_out`
  bool bank_done = !step_mode;                         // the live bank of this step has been handed out
  uint32_t bank_slot = (blockIdx.x * (uint32_t)NW + (uint32_t)wid) % max(A.n_slots, 1u), bank_probes = 0u;
  uint32_t res_next = 0u, res_end = 0u;                // records of bank_slot's bank reserved by this warp, not yet taken
  enum { BANK_CHUNK = 128 };
  if (step_mode && !A.step_source) src_exhausted = true;
  uint32_t n_seg = 0u;                                 // segments of this warp (warp-uniform)
  double acc_popw = 0.0;                               // census-step mode: weight this lane saw arrive at census A.step_k
  enum { W_COLL = 0, W_CHILDREN, W_LOST, W_SRC, W_CAP, W_FIS };   // (W_CAP, W_FIS: analog runs, where ledger entries are counts)
#define WCNT(k, v) do { const uint32_t v__ = (v); if (lane == 0 && v__ != 0u) sh.wcnt[wid][k] += v__; } while (0)

  for (;;) {
    // A refill leaves `pool_reserve` slots free: fission children are born into the parent's pool, and a pool that
    // refills to the brim sends them through the global queue in HBM instead (measured: 16 warps x 88 slots filled
    // completely ran 1.7x slower than 104 slots, 64 slots 6x slower -- profiles/r02b).  A refill that cannot fill
    // half a warp waits while the pool has other work.
    const uint32_t room = nFree > A.pool_reserve ? nFree - A.pool_reserve : 0u;
    int phase;                                         // 0 = R, 1 = F, 2 = C
    if (nF >= 32u) phase = 1;
    else if (nC >= 32u) phase = 2;
    else if (room >= (step_mode ? 32u : 16u) && dry == 0u) phase = 0;   // (bank refills come in full rounds)
    else if (nF > 0u && nF >= nC) phase = 1;
    else if (nC > 0u) phase = 2;
    else phase = 0;
    if (dry) --dry;

    if (phase == 0) {
      // =============== R: acquire work for up to 32 free slots, initialise the new particles (A.3, A.6) ===============
      const uint32_t want = min(32u, max(room, 1u));   // (room = 0 only with an empty pool smaller than the reserve)
      if (step_mode && !bank_done) {
        // ---- census-step mode: particles of the live bank first (full records: nothing is sampled here) ----
        // The warp reserves BANK_CHUNK records of the current batch slot's bank with one global atomic and asks for them
        // in L2; its refills then take up to 32 of them at a time.  (One returning atomic and one trip to DRAM per
        // refill were a quarter of the warp time of a census-step launch, profiles/r02d.)
        if (res_next == res_end) {
          uint32_t rb = 0u, cnt = 0u;
          if (lane == 0) { cnt = min(A.in.count[bank_slot], A.bank_cap); rb = atomicAdd(A.in.cursor + bank_slot, (uint32_t)BANK_CHUNK); }
          rb = __shfl_sync(MCDC_FULL, rb, 0); cnt = __shfl_sync(MCDC_FULL, cnt, 0);
          if (rb >= cnt) {                               // this batch slot is handed out: try the next one
            bank_slot = (bank_slot + 1u) % A.n_slots;
            if (++bank_probes >= A.n_slots) bank_done = true;
            continue;
          }
          bank_probes = 0u;
          res_next = rb; res_end = min(rb + (uint32_t)BANK_CHUNK, cnt);
          for (uint32_t r = res_next + 32u + (uint32_t)lane; r < res_end; r += 32u) {   // (the first 32 are loaded right below)
            const size_t j = (size_t)bank_slot * A.bank_cap + r;
            prefetch_l2(A.in.x + j); prefetch_l2(A.in.y + j); prefetch_l2(A.in.z + j); prefetch_l2(A.in.t + j);
            prefetch_l2(A.in.w + j); prefetch_l2(A.in.key + j); prefetch_l2(A.in.meta + j);
            if (!gen_mode) { prefetch_l2(A.in.ux + j); prefetch_l2(A.in.uy + j); prefetch_l2(A.in.uz + j); }
          }
        }
        const uint32_t base = res_next;
        const uint32_t nb = min(want, res_end - res_next);
        res_next += nb;
        const bool actb = (uint32_t)lane < nb;
        unsigned long long bkey = 0ull;
        uint32_t bctr = 0u, bgi = 0u;
        bool live = false;
        unsigned m_live = 0u;
        if (actb && gen_mode) {                          // a birth record: group and direction are sampled in the C phase
          const uint32_t i = (uint32_t)PL(L_FREE, lb + nFree - 1u - (uint32_t)lane), gi = lb + i;
          const size_t j = (size_t)bank_slot * A.bank_cap + base + (uint32_t)lane;
          const int4 m = A.in.meta[j];                   // {cell, -, counter, -}
          PD(D_X, gi) = A.in.x[j]; PD(D_Y, gi) = A.in.y[j]; PD(D_Z, gi) = A.in.z[j]; PD(D_T, gi) = A.in.t[j];
          PW(gi) = A.in.w[j];
          PK(gi) = A.in.key[j]; PU(U_CTR, gi) = (uint32_t)m.z;
          PU(U_CL, gi) = (uint32_t)m.x | (NONE16 << 16);
          PU(U_META, gi) = 255u | ((uint32_t)A.step_k << 8) | (bank_slot << 20);
          if (RECORD) PU(U_HID, gi) = A.in.hid[j];
          PL(L_C, lb + nC + (uint32_t)lane) = (uint8_t)i;
          bkey = A.in.key[j]; bctr = (uint32_t)m.z; bgi = gi;
        } else if (!gen_mode) {
          // (a record that the in-place population control removed is a hole, cell = -1: it takes no slot)
          const size_t j = (size_t)bank_slot * A.bank_cap + base + (uint32_t)(actb ? lane : 0);
          const int4 m = A.in.meta[j];                   // {cell, last surface, counter, group}
          live = actb && m.x >= 0;
          m_live = __ballot_sync(MCDC_FULL, live);
        }
        if (live) {
          const uint32_t rk = lanes_below(m_live, lane);
          const uint32_t i = (uint32_t)PL(L_FREE, lb + nFree - 1u - rk), gi = lb + i;
          const size_t j = (size_t)bank_slot * A.bank_cap + base + (uint32_t)lane;
          const double ux = A.in.ux[j], uy = A.in.uy[j], uz = A.in.uz[j];
          const int4 m = A.in.meta[j];
          PD(D_X, gi) = A.in.x[j]; PD(D_Y, gi) = A.in.y[j]; PD(D_Z, gi) = A.in.z[j]; PD(D_T, gi) = A.in.t[j];
          PD(D_UX, gi) = ux; PD(D_UY, gi) = uy; PD(D_UZ, gi) = uz;
          PD(D_IX, gi) = 1.0 / ux; PD(D_IY, gi) = 1.0 / uy; PD(D_IZ, gi) = 1.0 / uz;
          PW(gi) = A.in.w[j];
          PK(gi) = A.in.key[j]; PU(U_CTR, gi) = (uint32_t)m.z;
          PU(U_CL, gi) = (uint32_t)m.x | ((m.y < 0 ? NONE16 : (uint32_t)m.y) << 16);
          PU(U_META, gi) = (uint32_t)m.w | ((uint32_t)A.step_k << 8) | (bank_slot << 20);
          if (RECORD) PU(U_HID, gi) = A.in.hid[j];
          PL(L_F, lb + nF + rk) = (uint8_t)i;
          bkey = A.in.key[j]; bctr = (uint32_t)m.z; bgi = gi;
        }
        // a record that comes back with an odd counter needs the second half of its current block again
        if (__any_sync(MCDC_FULL, (bctr & 1u) != 0u)) {
          const ulonglong2 blk = philox_block(bkey, bctr >> 1);
          if (bctr & 1u) PC(bgi) = blk.y;
        }
        if (gen_mode) { nFree -= nb; nC += nb; }
        else { const uint32_t nl = (uint32_t)__popc(m_live); nFree -= nl; nF += nl; }
        __syncwarp();
        continue;
      }
      // source histories come from the warp's own chunk of the sub-batch; one global atomic per chunk
      // Chunks are dealt round-robin over the batch slots, so the warps in flight spread their scores over all the
      // slot accumulators instead of contending for the hot bins of one.
      while (src_next == src_end && !src_exhausted) {   // (a ragged last slot can yield an empty chunk)
        uint32_t ci = 0u;
        if (lane == 0) ci = atomicAdd(A.hist_cursor, 1u);
        ci = __shfl_sync(MCDC_FULL, ci, 0);
        if (ci >= A.n_chunks) src_exhausted = true;
        else {
          const uint32_t slot = ci % A.n_slots, j = ci / A.n_slots;
          const unsigned long long lo = (unsigned long long)slot * A.hb + (unsigned long long)j * A.src_chunk;
          const unsigned long long hi = min(min(lo + A.src_chunk, (unsigned long long)(slot + 1u) * A.hb), (unsigned long long)A.n_hist);
          src_next = (uint32_t)min(lo, hi); src_end = (uint32_t)hi;
        }
      }
      const uint32_t n_src = min(want, src_end - src_next), src_base = src_next;
      src_next += n_src;
      const bool src_done = src_exhausted && src_next == src_end;
      // the global queue only holds children that did not fit their parent's pool: look at it when this warp has
      // no source left, and now and then otherwise
      uint32_t got = 0u;
      unsigned long long qbase = 0ull;
      int flags = 0;                                   // 1 = abort (overflow flagged), 4 = queue empty
      if (n_src < want && (src_done || (r_calls & 15u) == 0u)) {
        if (lane == 0) {
          if (*(volatile int *)&A.cnt->overflow) flags |= 1;
          const unsigned long long h = ld_volatile_u64(q_head), t = ld_volatile_u64(q_tail);
          if (t > h) {
            const unsigned long long w = min((unsigned long long)(want - n_src), t - h);
            if (atomicCAS(q_head, h, h + w) == h) { got = (uint32_t)w; qbase = h; }
          } else flags |= 4;
        }
        flags = __shfl_sync(MCDC_FULL, flags, 0);
        got = __shfl_sync(MCDC_FULL, got, 0);
        qbase = __shfl_sync(MCDC_FULL, qbase, 0);
      }
      ++r_calls;
      if (flags & 1) break;                            // a queue overflow was flagged somewhere: the run is void
      const uint32_t total = got + n_src;
      if (total == 0u) {
        if (nF == 0u && nC == 0u) {
          if (src_done && (flags & 4)) break;          // pool empty, no source left, queue empty
          __nanosleep(256);
        } else dry = 8u;                               // nothing to take right now: work on what the pool holds
        continue;
      }
      const bool act = (uint32_t)lane < total;
      const uint32_t i = act ? (uint32_t)PL(L_FREE, lb + nFree - 1u - (uint32_t)lane) : 0u;
      nFree -= total;
      double x = 0.0, y = 0.0, z = 0.0, t = 0.0, w = 1.0;
      unsigned long long key = 0ull;
      uint32_t ctr = 0u, hid = 0u, slot = 0u;
      int cell = 0, pk = 0;
      bool ok = act, is_src = false, skip = false;     // skip: a source born in another census step (census-step mode)
      if (act && (uint32_t)lane >= n_src) {            // a fission child from the global queue (A.6)
        const unsigned long long qi = qbase + (unsigned long long)((uint32_t)lane - n_src);
        const uint32_t j = (uint32_t)qi & A.q.mask;
        const uint32_t expect = (uint32_t)(qi + 1ull);
        for (uint32_t spin = 0; ld_acquire_u32(A.q.flag + j) != expect; ++spin) {
          if ((spin & 255u) == 255u && (*(volatile int *)&A.cnt->overflow || spin > (1u << 26))) {
            atomicExch(&A.cnt->overflow, 1);           // producer gave up (overflow) or never published
            ok = false;
            break;
          }
        }
        x = A.q.x[j]; y = A.q.y[j]; z = A.q.z[j]; t = A.q.t[j];
        if (WEIGHTED) w = A.q.w[j];
        key = A.q.key[j];
        const int4 m = A.q.meta[j];
        cell = ok ? m.x : 0; pk = m.y; hid = (uint32_t)m.z; slot = (uint32_t)m.w;
      } else if (act) {                                // a new source history (A.3): xi_x, xi_y, xi_z, xi_t
        is_src = true;
        hid = src_base + (uint32_t)lane;
        slot = hid / A.hb;
        key = mix64(A.seed_mixed ^ (A.first_history + (unsigned long long)hid));
        // xi_x, xi_y = block 0, xi_z, xi_t = block 1
        const ulonglong2 b0 = philox_block(key, 0u), b1 = philox_block(key, 1u);
        const double xi_x = u64_to_unit(b0.x), xi_y = u64_to_unit(b0.y), xi_z = u64_to_unit(b1.x), xi_t = u64_to_unit(b1.y);
        ctr = 4u;
        x = T.src_lo[0] + xi_x * (T.src_hi[0] - T.src_lo[0]);
        y = T.src_lo[1] + xi_y * (T.src_hi[1] - T.src_lo[1]);
        z = T.src_lo[2] + xi_z * (T.src_hi[2] - T.src_lo[2]);
        t = T.src_t0 + xi_t * (T.src_t1 - T.src_t0);
        pk = census_index(tb, t);
        if (step_mode && !A.step_single && pk != A.step_k) { skip = true; ok = false; }
      }
      // group: chi of the fission-site material (child) or the source pdf; then the direction.  The counter is even here
      // (4 after a source position, 0 for a child): xi_g, xi_mu = one block, xi_phi = the first half of the next, whose
      // second half is kept for the particle's next draw
      const ulonglong2 ba = philox_block(key, ctr >> 1), bb = philox_block(key, (ctr >> 1) + 1u);
      const double xi_g = u64_to_unit(ba.x);
      unsigned long long half = ba.y;                  // second half of the block the next draw falls in
      int g;
      if (is_src) g = sample_cdf([&](int q) { return tb.src_cdf(q); }, G, T.src_last, xi_g);
      else {
        const int mat = (int)((tb.template ldb<uint32_t>(T.o_cell2 + (uint32_t)cell * CELL2_BYTES + C2_INFO) >> 8) & 255u);
        g = sample_cdf([&](int q) { return tb.cdf_chi(mat * G + q); }, G, tb.last_chi(mat), xi_g);
      }
      double ux, uy, uz;
      if (is_src && T.src_dir_mode != 0) { ux = T.src_dir[0]; uy = T.src_dir[1]; uz = T.src_dir[2]; ctr += 1u; }
      else {
        isotropic(u64_to_unit(ba.y), u64_to_unit(bb.x), ux, uy, uz);
        ctr += 3u; half = bb.y;
      }
      if (is_src) {
        // (a point source proved to lie strictly inside one cell at create time skips the search: warp-uniform)
        const bool known = T.src_cell >= 0 &&
                           (!T.src_chk || (x > T.src_clo[0] && x < T.src_chi[0] && y > T.src_clo[1] && y < T.src_chi[1] &&
                                           z > T.src_clo[2] && z < T.src_chi[2]));
        cell = known ? T.src_cell : slow_locate_source<RGN>(gT, x, y, z, ux, uy, uz);
        if (cell < 0) ok = false;                      // a source particle outside every cell is lost (A.3)
      }
      const unsigned m_lost = __ballot_sync(MCDC_FULL, is_src && cell < 0 && !skip);
      if (m_lost) { WCNT(W_LOST, (uint32_t)__popc(m_lost)); if (lane == 0) atomicAdd(&sh.led[LED_LOST], (double)__popc(m_lost)); }
      if (step_mode) WCNT(W_SRC, (uint32_t)__popc(__ballot_sync(MCDC_FULL, is_src && !skip)));
      else WCNT(W_SRC, n_src);
      if (ok) {
        const uint32_t gi = lb + i;
        PP(P_XY, gi) = make_double2(x, y); PP(P_ZT, gi) = make_double2(z, t); PP(P_U01, gi) = make_double2(ux, uy);
        PP(P_U2I0, gi) = make_double2(uz, 1.0 / ux); PP(P_I12, gi) = make_double2(1.0 / uy, 1.0 / uz);
        if (WEIGHTED) PW(gi) = w;
        PKC(gi) = make_ulonglong2(key, half);
        PU(U_CTR, gi) = ctr; PU(U_CL, gi) = (uint32_t)cell | (NONE16 << 16);
        PU(U_META, gi) = (uint32_t)g | ((uint32_t)pk << 8) | (slot << 20);
        if (RECORD) PU(U_HID, gi) = hid;
      }
      const unsigned m_ok = __ballot_sync(MCDC_FULL, ok), m_bad = __ballot_sync(MCDC_FULL, act && !ok);
      if (ok) PL(L_F, lb + nF + lanes_below(m_ok, lane)) = (uint8_t)i;
      if (act && !ok) PL(L_FREE, lb + nFree + lanes_below(m_bad, lane)) = (uint8_t)i;
      nF += (uint32_t)__popc(m_ok); nFree += (uint32_t)__popc(m_bad);
      __syncwarp();
      continue;
    }

    if (phase == 1) do {
      // =============== F: one segment -- distances, event choice, score, move, census / surface event ===============
      // (a full flight round is followed by the next one without going through the phase choice again)
      const uint32_t n = min(32u, nF);
      nF -= n;
      n_seg += n;                                      // every lane of a flight round makes one segment
      const bool act = (uint32_t)lane < n;
      // (a round is almost always full; the idle lanes of a partial one read the slot of its last active lane, so that
      // no load below needs a guard or a default -- their results are dropped: ev = -1, stores and scores keep `act`)
      const uint32_t i = (uint32_t)PL(L_F, lb + nF + min((uint32_t)lane, n - 1u));
      const uint32_t gi = lb + i;
      // distance to collision first: the random-number state is dead before the geometry needs its registers
      uint32_t cl, meta;
      double d_coll;
      {
        const unsigned long long key = PK(gi);
        const uint32_t ctr = PU(U_CTR, gi);
        cl = PU(U_CL, gi); meta = PU(U_META, gi);
        // always consumed (D3).  Draw 2b is the first half of block b and leaves the second half in the pool for
        // draw 2b + 1, wherever that one is made (the collision phase reads it; here the block is computed for the
        // even lanes of the round anyway)
        const ulonglong2 blk = philox_block(key, ctr >> 1);
        const bool odd = (ctr & 1u) != 0u;
        const double xi = u64_to_unit(odd ? blk.y : blk.x);
        if (act) { PU(U_CTR, gi) = ctr + 1u; if (!odd) PC(gi) = blk.y; }
        // xi = (k + 1/2) 2^-52 lies in [2^-53, 1 - 2^-53]: telling the compiler so removes log's subnormal / zero / inf / NaN
        // paths (22 instructions of ~100) without touching the arithmetic of the ordinary one
        __builtin_assume(__double2hiint(xi) >= 0x3c900000 && __double2hiint(xi) < 0x3ff00000);
        d_coll = -log(xi);
      }
      const int cell = (int)(cl & 0xFFFFu), g = (int)(meta & 255u), pk = (int)((meta >> 8) & 4095u);
      const uint32_t last = cl >> 16;                  // surface the particle sits on, NONE16 if none
      const uint32_t rec = T.o_cell2 + (uint32_t)cell * CELL2_BYTES;
      const uint32_t info = tb.template ldb<uint32_t>(rec + C2_INFO);
      const int n_other = (int)(info & 255u), mg = (int)((info >> 8) & 255u) * G + g;
      d_coll *= tb.inv_sig_t(mg);                      // (1 / Sigma_t is +inf in a void: no collision)
      // 1/direction is kept in the pool (three divisions per segment otherwise)
      const double2 xy = PP(P_XY, gi), zt = PP(P_ZT, gi), u01 = PP(P_U01, gi), u2i0 = PP(P_U2I0, gi), i12 = PP(P_I12, gi);
      double x = xy.x, y = xy.y, z = zt.x, t = zt.y, ux = u01.x, uy = u01.y, uz = u2i0.x, ix = u2i0.y, iy = i12.x, iz = i12.y;
      // ---- faces: one candidate per axis, picked by the sign of the direction component ----
      // sign bit alone: for a component that is exactly +-0 the face distance is inf or NaN and is rejected below
      const bool px = __double2hiint(ux) >= 0, py = __double2hiint(uy) >= 0, pz = __double2hiint(uz) >= 0;
      const int fx = px ? 1 : 0, fy = py ? 3 : 2, fz = pz ? 5 : 4;
      const uint32_t sfx = tb.template ldb<uint16_t>(rec + C2_FACE_SURF + 2u * fx);
      const uint32_t sfy = tb.template ldb<uint16_t>(rec + C2_FACE_SURF + 2u * fy);
      const uint32_t sfz = tb.template ldb<uint16_t>(rec + C2_FACE_SURF + 2u * fz);
      // (a side without a face names a sentinel entry of the surface table: +inf above, -inf below)
      const double bx = tb.surf_q0((int)sfx), by = tb.surf_q0((int)sfy), bz = tb.surf_q0((int)sfz);
      const double dx = (bx - x) * ix, dy = (by - y) * iy, dz = (bz - z) * iz;   // 0 * inf = NaN: rejected below
      // nearest face; equal distances (an edge hit): the earlier half-space of the cell's list wins (D5)
      const bool vx = dx > 0.0 && dx < INF, vy = dy > 0.0 && dy < INF, vz = dz > 0.0 && dz < INF;
      double d_surf = vx ? dx : INF;
      int which = vx ? fx : -1;                        // 2*axis + side of the nearest face, 6 + j for other j
      if (vy && dy < d_surf) { d_surf = dy; which = fy; }
      if (vz && dz < d_surf) { d_surf = dz; which = fz; }
      // two faces at exactly the same finite distance: rare enough for a branch the whole warp takes or skips
      if (__any_sync(MCDC_FULL, (vx && vy && dx == dy) || (vz && (dz == dx || dz == dy) && (vx || vy)))) {
        d_surf = vx ? dx : INF; which = vx ? fx : -1;
        bool ty = vy && dy < d_surf;
        if (vy && dy == d_surf) ty = tb.template ldb<uint8_t>(rec + C2_FACE_IDX + fy) < tb.template ldb<uint8_t>(rec + C2_FACE_IDX + which);
        if (ty) { d_surf = dy; which = fy; }
        bool tz = vz && dz < d_surf;
        if (vz && dz == d_surf) tz = tb.template ldb<uint8_t>(rec + C2_FACE_IDX + fz) < tb.template ldb<uint8_t>(rec + C2_FACE_IDX + which);
        if (tz) { d_surf = dz; which = fz; }
      }
      // ---- other half-spaces (cylinders, general quadrics, redundant planes), list order, strict < ----
      const uint32_t orec = T.o_other2 + (info >> 16) * OTHER2_BYTES;
#pragma unroll 1                                       // (peeled, the loop left a second, cold copy of its body in the flight phase)
      for (int j = 0; j < n_other; ++j) {
        const uint2 e = tb.template ldb<uint2>(orec + (uint32_t)j * OTHER2_BYTES);
        const uint32_t s = e.x & 0xFFFFu;
        const int type = (int)((e.y >> 9) & 7u);
        double u;
        if (type == ST_CYL_Z) {
          const double2 q01 = tb.surf_q01((int)s);
          const double r2 = tb.surf_q23((int)s).x;
          const double ex = x - q01.x, ey = y - q01.y;
          u = quad_root_pos_a(ux * ux + uy * uy, ex * ux + ey * uy, (s == last) ? 0.0 : (ex * ex + ey * ey - r2));
        } else {
          u = slow_distance(gT, (int)s, type, s == last, x, y, z, ux, uy, uz);
        }
        if (u < d_surf) { d_surf = u; which = 6 + j; }
      }
      double w = 1.0;
      if (WEIGHTED) w = act ? PW(gi) : 0.0;
      const double t_census = tb.census(pk);
      const double d_time = tb.speed(g) * (t_census - t);
      int ev;
      double d;
      if (d_time <= d_surf && d_time <= d_coll) { d = d_time; ev = EV_CENSUS; }
      else if (d_surf <= d_coll) { d = d_surf; ev = EV_SURFACE; }
      else { d = d_coll; ev = EV_COLLISION; }
      if (!act) { ev = -1; d = 0.0; }
      // census-step mode: the arrivals of this round will be appended to their batch's census bank further down; the
      // counter is bumped here, one atomic per batch slot in the warp, so that its round trip overlaps the rest of the round
      unsigned park_peers = 0u;
      int park_leader = 0;
      uint32_t park_base = 0u;
      if (step_mode) {
        const bool park = act && ev == EV_CENSUS && pk != T.K - 1;
        if (__any_sync(MCDC_FULL, park)) {
          const int bslot = park ? (int)(meta >> 20) : -1;
          park_peers = __match_any_sync(MCDC_FULL, bslot);
          park_leader = __ffs(park_peers) - 1;
          if (park && lane == park_leader) park_base = atomicAdd(A.census_out.count + bslot, (uint32_t)__popc(park_peers));
        }
      }

      // ---- track-length score (A.7) from the pre-move state ----
      {
        const uint32_t slot = meta >> 20;
        TallySink S;
        S.slab = nullptr; S.global_x = A.x_acc + (size_t)slot * T.n_bins; S.slab_lo = 0; S.slab_bins = 0;
        S.aggregate = (SCORE == 0) ? A.aggregate : (SCORE == 2 ? 1 : 0);
        const uint32_t cbin = tb.template ldb<uint32_t>(rec + C2_BIN);
        const int tbin = tb.template ld<int>(T.o_tbin_k, pk);
        const bool one_bin = ONEBIN || (cbin != NONE32 && tbin >= 0);   // the whole segment lies in one tally bin
        if (!ONEBIN) {
          if (__any_sync(MCDC_FULL, act && !one_bin))
            general_score<STAGED>(T, S.global_x, A.aggregate, act && !one_bin, &PD(0, 0), N, gi, g, pk, d, w);
        }
        if (ONEBIN || __any_sync(MCDC_FULL, act && one_bin)) {
          const bool sc = act && one_bin && d > 0.0;
          if (SCORE == 1) {                            // one RED; the usual case indexes all accumulators with 32 bits
            if (sc) {
              if (bins32) red_add_f64(A.x_acc + (slot * (uint32_t)T.n_bins + (uint32_t)((tbin * G + g) * (int)n_spatial + (int)cbin)), WEIGHTED ? w * d : d);
              else red_add_f64(S.global_x + ((long long)(tbin * G + g) * n_spatial + (long long)cbin), WEIGHTED ? w * d : d);
            }
          } else {
            long long bin = -1;
            if (sc) bin = (long long)(tbin * G + g) * n_spatial + (long long)cbin;
            tally_add_converged(S, bin, WEIGHTED ? w * d : d);
          }
        }
      }
      // ---- move (A.3) ----
      x += d * ux; y += d * uy; z += d * uz;
      t = (ev == EV_CENSUS) ? t_census : t + d * tb.inv_speed(g);
      bool alive = act;
      uint32_t new_cl = cl;
      int census_k = -1;
      if (ev == EV_CENSUS) {                           // A.8: bookkeeping only, then the next interval
        census_k = pk;
        if (d > 0.0) new_cl = (cl & 0xFFFFu) | (NONE16 << 16);
        if (pk == T.K - 1 || step_mode) alive = false;   // census-step mode: parked in the census bank below
        else meta += 1u << 8;
      } else if (ev == EV_SURFACE) {                   // A.5
        const bool is_face = which < 6;
        const int wf = is_face ? which : 0, jo = is_face ? 0 : which - 6;
        const uint2 e = tb.template ldb<uint2>(orec + (uint32_t)jo * OTHER2_BYTES);
        const uint32_t nb_f = tb.template ldb<uint16_t>(rec + C2_FACE_NB + 2u * wf);
        const uint32_t bc_f = (tb.template ldb<uint16_t>(rec + C2_FACE_BC) >> (2 * wf)) & 3u;
        const uint32_t s_f = (which == fx) ? sfx : ((which == fy) ? sfy : sfz);
        const uint32_t s_star = is_face ? s_f : (e.x & 0xFFFFu), nb = is_face ? nb_f : (e.x >> 16);
        const int bc = (int)(is_face ? bc_f : ((e.y >> 12) & 3u));
        const int type = is_face ? (which >> 1) : (int)((e.y >> 9) & 7u);   // faces: ST_PLANE_X/Y/Z = axis
        int idx = is_face ? -1 : (int)(e.y & 255u);
        new_cl = (cl & 0xFFFFu) | (s_star << 16);
        if (bc == 1) {                                 // vacuum: leaks
          alive = false;
          if (WEIGHTED) atomicAdd(&sh.wled[wid][LED_LEAK], w); else atomicAdd(&sh.n_leak, 1u);
        } else if (bc == 2) {                          // reflective: specular, stays in the cell
          if (type == ST_PLANE_X) { PD(D_UX, gi) = -ux; PD(D_IX, gi) = -ix; }
          else if (type == ST_PLANE_Y) { PD(D_UY, gi) = -uy; PD(D_IY, gi) = -iy; }
          else if (type == ST_PLANE_Z) { PD(D_UZ, gi) = -uz; PD(D_IZ, gi) = -iz; }
          else {
            double u3[3] = {ux, uy, uz};
            slow_reflect(gT, (int)s_star, type, x, y, z, u3);
            PD(D_UX, gi) = u3[0]; PD(D_UY, gi) = u3[1]; PD(D_UZ, gi) = u3[2];
            PD(D_IX, gi) = 1.0 / u3[0]; PD(D_IY, gi) = 1.0 / u3[1]; PD(D_IZ, gi) = 1.0 / u3[2];
          }
        } else {                                       // transmission: the cell on the other side
          // a certified neighbour holds every point of this surface patch that lies strictly inside the cell's
          // forward faces (mcdc_host.cu); anything else takes the full search of A.5
          const int ax = (which < 6) ? (which >> 1) : -1;
          // (x < bx going up, x > bx going down: bx - x has the sign of 1 / ux and is not zero; a sentinel bx = +-inf passes)
          const bool in_x = ax == 0 || (bx - x) * ix > 0.0;
          const bool in_y = ax == 1 || (by - y) * iy > 0.0;
          const bool in_z = ax == 2 || (bz - z) * iz > 0.0;
          int c2;
          if (nb != NONE16 && in_x && in_y && in_z) c2 = (int)nb;
          else {
            if (idx < 0) idx = (int)tb.template ldb<uint8_t>(rec + C2_FACE_IDX + which);
            c2 = slow_cross<RGN>(gT, cell, idx, (int)s_star, x, y, z, ux, uy, uz);
          }
          if (c2 < 0) { alive = false; atomicAdd(&sh.led[LED_LOST], w); atomicAdd(&sh.wcnt[wid][W_LOST], 1u); }   // (never, in a sound geometry)
          else new_cl = (uint32_t)c2 | (s_star << 16);
        }
      }
      if (act) {
        PP(P_XY, gi) = make_double2(x, y); PP(P_ZT, gi) = make_double2(z, t);
        if (new_cl != cl) PU(U_CL, gi) = new_cl;
        if (ev == EV_CENSUS) PU(U_META, gi) = meta;
        if (RECORD && ev != EV_COLLISION) atomicAdd(A.ev + (size_t)PU(U_HID, gi) * 4 + (ev == EV_CENSUS ? 3 : 1), 1u);
      }
      if (step_mode) {
        // ---- census-step mode: park the arrivals of a census that is not the last in their batch's census bank ----
        const bool park = act && ev == EV_CENSUS && pk != T.K - 1;
        if (__any_sync(MCDC_FULL, park)) {
          const int bslot = park ? (int)(meta >> 20) : -1;
          const uint32_t idx = __shfl_sync(MCDC_FULL, park_base, park_leader) + lanes_below(park_peers, lane);
          if (park) {
            if (idx >= A.bank_cap) atomicExch(&A.cnt->overflow, 1);
            else {
              const size_t j = (size_t)bslot * A.bank_cap + idx;
              const Bank &O = A.census_out;
              const uint32_t last2 = new_cl >> 16;
              O.x[j] = x; O.y[j] = y; O.z[j] = z; O.ux[j] = ux; O.uy[j] = uy; O.uz[j] = uz; O.t[j] = t; O.w[j] = w;
              O.key[j] = PK(gi); O.hid[j] = RECORD ? PU(U_HID, gi) : 0u;
              O.meta[j] = make_int4(cell, last2 == NONE16 ? -1 : (int)last2, (int)PU(U_CTR, gi), g);
            }
          }
        }
      }
      // ---- census population (A.8) ----
      // Asynchronous modes: one native shared-memory add per arriving lane (the hardware serialises equal addresses; a
      // __match_any_sync to merge them first cost more than it saved).  Census-step mode: every arrival of the launch
      // carries the index A.step_k, so the count is one ballot and the weight is summed in a register until the end
      // (lanes adding to the same shared-memory DOUBLE serialise in a compare-and-swap loop: that add was 56 % of the
      // samples of a census-step launch, profiles/r02c).  The final-census ledger entry is what reached the last census:
      // it is taken from that sum when the block ends.
      if (step_mode) {
        const unsigned m_cen = __ballot_sync(MCDC_FULL, census_k >= 0);
        if (m_cen && lane == 0) atomicAdd(s_popn + A.step_k, (uint32_t)__popc(m_cen));
        if (WEIGHTED && census_k >= 0) acc_popw += w;
      } else if (census_k >= 0) {
        atomicAdd(s_popn + census_k, 1u);
        if (WEIGHTED) {
          atomicAdd(s_popw + (lane & (POPW_COPIES - 1)) * T.K + census_k, w);   // (copies: see POPW_COPIES)
        }
      }
      // (surface events are not counted here: segments - collisions - census events, at the end of the block)
      // ---- hand the slots on: F again, C, or FREE ----
      const bool toF = alive && ev != EV_COLLISION, toC = alive && ev == EV_COLLISION, dead = act && !alive;
      const unsigned mF = __ballot_sync(MCDC_FULL, toF), mC = __ballot_sync(MCDC_FULL, toC), mD = __ballot_sync(MCDC_FULL, dead);
      if (toF) PL(L_F, lb + nF + lanes_below(mF, lane)) = (uint8_t)i;
      if (toC) PL(L_C, lb + nC + lanes_below(mC, lane)) = (uint8_t)i;
      if (dead) PL(L_FREE, lb + nFree + lanes_below(mD, lane)) = (uint8_t)i;
      nF += (uint32_t)__popc(mF); nC += (uint32_t)__popc(mC); nFree += (uint32_t)__popc(mD);
      __syncwarp();
    } while (nF >= 32u);
    if (phase == 1) continue;

    // =============== C: collisions (A.6) ===============
    {
      const uint32_t n = min(32u, nC);
      nC -= n;
      const bool act = (uint32_t)lane < n;
      // (idle lanes of a partial round read the slot of its last active lane, as in the flight phase: no guarded loads)
      const uint32_t i = (uint32_t)PL(L_C, lb + nC + min((uint32_t)lane, n - 1u));
      const uint32_t gi = lb + i;
      const ulonglong2 kc = PKC(gi);
      const unsigned long long key = kc.x;
      unsigned long long r0 = kc.y;                    // the half block the pool kept (used when the counter is odd)
      const uint32_t ctr = PU(U_CTR, gi), cl = PU(U_CL, gi), meta = PU(U_META, gi);
      const int cell = (int)(cl & 0xFFFFu);
      int g = (int)(meta & 255u);
      const bool born = act && g == 255;               // a fission child placed in this pool: only its flight is sampled
      if (g == 255) g = 0;
      const int mat = (int)((tb.template ldb<uint32_t>(T.o_cell2 + (uint32_t)cell * CELL2_BYTES + C2_INFO) >> 8) & 255u);
      const int mg = mat * G + g;
      // The random numbers of this round.  A collision consumes at most four draws from the counter c it arrives with
      // (reaction, group, mu, phi; a fission: reaction, nu -- its children draw from streams of their own in a later
      // round; a child: group, mu, phi), five with a weight roulette.  Draws c .. c+3 lie in the blocks b0 = (c+1) >> 1
      // and b0 + 1, plus -- when c is odd -- the half block the pool kept from the draw before (PC): two Philox blocks
      // per round whatever the lanes do (Appendix B allows caching the unused half block; the draws are the same).
      const bool odd = (ctr & 1u) != 0u;
      const uint32_t b0 = (ctr + 1u) >> 1;
      unsigned long long r1, r2, r3, r4 = 0ull;
      {
        const ulonglong2 ba = philox_block(key, b0), bb = philox_block(key, b0 + 1u);
        r1 = odd ? ba.x : ba.y; r2 = odd ? ba.y : bb.x; r3 = odd ? bb.x : bb.y;
        if (!odd) r0 = ba.x; else r4 = bb.y;
      }
      const double xi_r = u64_to_unit(r0);
      int kind = FI_NONE, n_child = 0;                 // kind of the outgoing flight; children of a fission
      bool alive = false, captured = false, fissioned = false, reborn = false, rouletted = false;
      uint32_t c0 = 0u;
      double w = 1.0, l_cap = 0.0, l_fis = 0.0, l_prod = 0.0, l_gain = 0.0, l_loss = 0.0;   // WEIGHTED only
      if (WEIGHTED) w = act ? PW(gi) : 0.0;
      // Appendix I: collision estimator, arriving weight.  Out of line: inlined, its ~150 instructions sat in the middle
      // of the C phase and cost runs that never enable the tally 8 % (profiles/r01f)
      if (WEIGHTED && A.xc_acc != nullptr && act && !born)
        slow_score_collision(gT, A.xc_acc + (size_t)(meta >> 20) * T.n_bins, PD(D_X, gi), PD(D_Y, gi), PD(D_Z, gi), PD(D_T, gi), g, w, mg);
      if (born) { kind = FI_CHILD; alive = true; }
      else if (act) {
        const double s_tot = tb.sig_s_tot(mg), sig_f = tb.sig_f(mg);
        bool scatter = false, dead = false;
        if (WEIGHTED && T.implicit_capture) {          // G.1: the captured fraction leaves the weight
          const double w_c = w * tb.cap_frac(mg);
          l_cap += w_c; w -= w_c;
          const double s_r = s_tot + sig_f;
          if (!(s_r > 0.0)) { l_cap += w; w = 0.0; dead = true; }
          else scatter = (xi_r * s_r < s_tot) || sig_f == 0.0;
        } else {
          const double yv = xi_r * tb.sig_t(mg);
          scatter = yv < s_tot;
          if (!scatter && (yv < tb.sig_sc(mg) || sig_f == 0.0)) { dead = true; captured = true; l_cap += w; }
        }
        if (dead) {
        } else if (scatter) {
          if (WEIGHTED && T.wr_threshold > 0.0 && w < T.wr_threshold) {   // G.2 weight roulette
            const double xi_w = u64_to_unit(r1);
            rouletted = true;
            if (xi_w * T.wr_survive < w) { l_gain += T.wr_survive - w; w = T.wr_survive; kind = FI_SCATTER; alive = true; }
            else l_loss += w;
          } else { kind = FI_SCATTER; alive = true; }
        } else {
          const double xi_nu = u64_to_unit(r1);
          n_child = (int)floor(tb.nu(mg) + xi_nu);
          c0 = ctr + 2u;
          fissioned = true;
          l_fis += w; l_prod += (double)n_child * w;
          if (n_child > 0 && !gen_mode) reborn = true;   // the parent's slot goes on as its first child (below)
        }
      }
      {
        const unsigned m_cap = __ballot_sync(MCDC_FULL, captured), m_fis = __ballot_sync(MCDC_FULL, fissioned);
        if (WEIGHTED) {
          // (each warp sum is 15 instructions: only the entries that some lane of this round touched are summed)
          if (__any_sync(MCDC_FULL, l_cap != 0.0)) { l_cap = warp_sum(l_cap); if (lane == 0) sh.wled[wid][LED_CAPTURE] += l_cap; }
          if (m_fis) {
            l_fis = warp_sum(l_fis); l_prod = warp_sum(l_prod);
            if (lane == 0) { sh.wled[wid][LED_FISSION_ABS] += l_fis; sh.wled[wid][LED_PRODUCTION] += l_prod; }
          }
          if (__any_sync(MCDC_FULL, rouletted)) {
            l_gain = warp_sum(l_gain); l_loss = warp_sum(l_loss);
            if (lane == 0) { sh.wled[wid][LED_VR_GAIN] += l_gain; sh.wled[wid][LED_VR_LOSS] += l_loss; }
          }
        } else WCNT(W_CAP, (uint32_t)__popc(m_cap));    // unit weights: captures, absorptions and production are counts
        if (m_fis) {
          const uint32_t kids = __reduce_add_sync(MCDC_FULL, (uint32_t)n_child);
          if (!WEIGHTED) WCNT(W_FIS, (uint32_t)__popc(m_fis));
          WCNT(W_CHILDREN, kids);
        }
        WCNT(W_COLL, (uint32_t)__popc(__ballot_sync(MCDC_FULL, act && !born)));
      }
      if (RECORD && act && !born) {
        atomicAdd(A.ev + (size_t)PU(U_HID, gi) * 4 + 0, 1u);
        if (n_child > 0) atomicAdd(A.ev + (size_t)PU(U_HID, gi) * 4 + 2, (uint32_t)n_child);
      }
      // fission: children 1..n-1 go to free slots of this pool (or the global queue), the parent's slot becomes child 0;
      // all of them are "born" entries of the C stack: a later round samples their group and direction
      // (generation mode: every child goes to the fission bank of the generation and the parent ends here)
      const int n_push = gen_mode ? n_child : ((n_child > 1) ? n_child - 1 : 0);
      if (__ballot_sync(MCDC_FULL, n_push > 0) != 0u) {
        int pre = n_push;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int v = __shfl_up_sync(MCDC_FULL, pre, o);
          if (lane >= o) pre += v;
        }
        const int total = __shfl_sync(MCDC_FULL, pre, 31);
        if (gen_mode) {
          uint32_t base = 0u;
          if (lane == 0) base = atomicAdd(A.census_out.count, (uint32_t)total);   // one batch slot in this mode
          base = __shfl_sync(MCDC_FULL, base, 0) + (uint32_t)(pre - n_push);
          if (n_push > 0) {
            const double x = PD(D_X, gi), y = PD(D_Y, gi), z = PD(D_Z, gi), t = PD(D_T, gi);
            const Bank &O = A.census_out;
            for (int c = 0; c < n_push; ++c) {
              const uint32_t j = base + (uint32_t)c;
              if (j >= A.bank_cap) { atomicExch(&A.cnt->overflow, 1); break; }
              O.x[j] = x; O.y[j] = y; O.z[j] = z; O.t[j] = t; O.w[j] = w;
              O.key[j] = child_key(key, c0, (uint32_t)c);
              O.meta[j] = make_int4(cell, -1, 0, 0);
              O.hid[j] = RECORD ? PU(U_HID, gi) : 0u;
            }
          }
        } else if ((uint32_t)total <= nFree) {         // the children fit this warp's pool: they join its C stack
          if (n_push > 0) {
            const double2 xy = PP(P_XY, gi), zt = PP(P_ZT, gi);
#pragma unroll 1
            for (int c = 0; c < n_push; ++c) {
              const uint32_t r = (uint32_t)(pre - n_push + c);
              const uint32_t i2 = (uint32_t)PL(L_FREE, lb + nFree - 1u - r), g2 = lb + i2;
              PP(P_XY, g2) = xy; PP(P_ZT, g2) = zt;
              if (WEIGHTED) PW(g2) = w;
              PK(g2) = child_key(key, c0, (uint32_t)(c + 1)); PU(U_CTR, g2) = 0u;
              PU(U_CL, g2) = (cl & 0xFFFFu) | (NONE16 << 16);
              PU(U_META, g2) = (meta & ~255u) | 255u;
              if (RECORD) PU(U_HID, g2) = PU(U_HID, gi);
              PL(L_C, lb + nC + r) = (uint8_t)i2;
            }
          }
          nFree -= (uint32_t)total; nC += (uint32_t)total;
        } else {                                       // pool full: publish them to the global queue (rare: out of line)
          double x = 0.0, y = 0.0, z = 0.0, t = 0.0;
          int4 qm = make_int4(0, 0, 0, 0);
          if (n_push > 0) {
            x = PD(D_X, gi); y = PD(D_Y, gi); z = PD(D_Z, gi); t = PD(D_T, gi);
            qm = make_int4(cell, (int)((meta >> 8) & 4095u), RECORD ? (int)PU(U_HID, gi) : 0, (int)(meta >> 20));
          }
          slow_publish_children(A.q, A.cnt, WEIGHTED, x, y, z, t, w, key, c0, n_push, pre, total, qm);
        }
      }
      if (reborn) {                                    // fission parent -> its first child, in place, born next round
        PK(gi) = child_key(key, c0, 0u); PU(U_CTR, gi) = 0u;
        PU(U_CL, gi) = (cl & 0xFFFFu) | (NONE16 << 16);
        PU(U_META, gi) = meta | 255u;
        if (WEIGHTED) PW(gi) = w;
      }
      // group and direction of the outgoing flight (A.6): one draw for the group, two for the direction
      if (__any_sync(MCDC_FULL, alive)) {
        // a scattered particle is past the reaction draw: group, mu, phi = draws c+1 .. c+3, and an odd c leaves draw
        // c+4 (r4, the second half of block b0+1) for later; a child starts at its counter: draws c .. c+2, an even c
        // leaves c+3 (r3)
        unsigned long long q_g = r1, q_mu = r2, q_phi = r3, half = r4;
        uint32_t used = 4u;
        if (born) { q_g = r0; q_mu = r1; q_phi = r2; half = r3; used = 3u; }
        if (WEIGHTED && __any_sync(MCDC_FULL, rouletted && alive)) {   // the roulette took draw c+1: one draw further
          const ulonglong2 bc = philox_block(key, b0 + 2u);
          if (rouletted) { q_g = r2; q_mu = r3; q_phi = odd ? r4 : bc.x; half = bc.y; used = 5u; }
        }
        const double xi_g = u64_to_unit(q_g);
        if (kind == FI_SCATTER) g = sample_cdf([&](int q) { return tb.cdf_s(mg * G + q); }, G, tb.last_s(mg), xi_g * tb.sig_s_tot(mg));
        else g = sample_cdf([&](int q) { return tb.cdf_chi(mat * G + q); }, G, tb.last_chi(mat), xi_g);
        double ux, uy, uz;
        isotropic(u64_to_unit(q_mu), u64_to_unit(q_phi), ux, uy, uz);
        if (alive) {
          PP(P_U01, gi) = make_double2(ux, uy); PP(P_U2I0, gi) = make_double2(uz, 1.0 / ux);
          PP(P_I12, gi) = make_double2(1.0 / uy, 1.0 / uz);
          if (WEIGHTED) PW(gi) = w;
          const uint32_t ctr_out = ctr + used;
          PU(U_CTR, gi) = ctr_out;
          if (ctr_out & 1u) PC(gi) = half;             // in the middle of a block: keep its second half for the next draw
          PU(U_META, gi) = (meta & ~255u) | (uint32_t)g;
          PU(U_CL, gi) = (cl & 0xFFFFu) | (NONE16 << 16);
        }
      }
      const unsigned mF = __ballot_sync(MCDC_FULL, alive), mC = __ballot_sync(MCDC_FULL, reborn), mD = __ballot_sync(MCDC_FULL, act && !alive && !reborn);
      if (alive) PL(L_F, lb + nF + lanes_below(mF, lane)) = (uint8_t)i;
      if (reborn) PL(L_C, lb + nC + lanes_below(mC, lane)) = (uint8_t)i;
      if (act && !alive && !reborn) PL(L_FREE, lb + nFree + lanes_below(mD, lane)) = (uint8_t)i;
      nF += (uint32_t)__popc(mF); nC += (uint32_t)__popc(mC); nFree += (uint32_t)__popc(mD);
      __syncwarp();
    }
  }

  // ---- warp totals -> block totals -> global ----
  __syncwarp();
  if (WEIGHTED && step_mode) {
    const double s = warp_sum(acc_popw);
    if (lane == 0 && s != 0.0) {
      atomicAdd(s_popw + A.step_k, s);
    }
  }
  if (lane == 0) {
    const uint32_t *wc = sh.wcnt[wid];
    atomicAdd(&sh.n_coll, (unsigned long long)wc[W_COLL]); atomicAdd(&sh.n_seg, (unsigned long long)n_seg);
    atomicAdd(&sh.n_children, (unsigned long long)wc[W_CHILDREN]);
    if (WEIGHTED) {
      for (int e = 0; e < LED_N; ++e)
        if (sh.wled[wid][e] != 0.0) atomicAdd(&sh.led[e], sh.wled[wid][e]);
    } else {                                             // the analog ledger, from the warp's counts
      if (wc[W_CAP]) atomicAdd(&sh.led[LED_CAPTURE], (double)wc[W_CAP]);
      if (wc[W_FIS]) atomicAdd(&sh.led[LED_FISSION_ABS], (double)wc[W_FIS]);
      if (wc[W_CHILDREN]) atomicAdd(&sh.led[LED_PRODUCTION], (double)wc[W_CHILDREN]);
    }
    atomicAdd(&sh.n_lost, (unsigned long long)wc[W_LOST]); atomicAdd(&sh.n_src, (unsigned long long)wc[W_SRC]);
  }
  __syncthreads();
  for (int k = tid; k < T.K; k += NT) {
    if (s_popn[k] != 0u) {
      double pw = (double)s_popn[k];
      if (WEIGHTED) { pw = 0.0; for (int c = 0; c < popw_copies(VARIANT); ++c) pw += s_popw[c * T.K + k]; }
      atomicAdd(A.pop_w + k, pw); atomicAdd(A.pop_n + k, (unsigned long long)s_popn[k]);
      atomicAdd(&sh.n_census, (unsigned long long)s_popn[k]);   // census events of the block = its population counts
      if (k == T.K - 1) atomicAdd(&sh.led[LED_CENSUS_FINAL], pw);   // what reached the last census is the final-census ledger entry
    }
  }
  __syncthreads();
  if (tid == 0) {
    DevCounters *cnt = A.cnt;
    if (!WEIGHTED) sh.led[LED_LEAK] += (double)sh.n_leak;
    for (int e = 0; e < LED_N; ++e)
      if (sh.led[e] != 0.0) atomicAdd(&cnt->ledger[1 + e], sh.led[e]);
    atomicAdd(&cnt->ledger[0], (double)sh.n_src);
    atomicAdd(&cnt->n[0], sh.n_src);
    atomicAdd(&cnt->n[1], sh.n_seg);
    atomicAdd(&cnt->n[2], sh.n_coll);
    atomicAdd(&cnt->n[3], sh.n_seg - sh.n_coll - sh.n_census);   // a segment ends in a collision, a census or a surface event
    atomicAdd(&cnt->n[4], sh.n_census);
    atomicAdd(&cnt->n[5], sh.n_children);
    atomicAdd(&cnt->n[6], sh.n_lost);
  }
}

#undef PD
#undef PK
#undef PC
#undef PP
#undef PKC
#undef PW
#undef PU
#undef PL
#undef WCNT

}  // namespace mcdc
