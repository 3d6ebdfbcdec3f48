// mcdc_pool.cuh -- k_pool: the event-based history kernel (default scheduler, MCDC_SCHED_ASYNC).
//
// Replaces the paper's Harmonize runtime ("segregating them into like-operations ... executed
// together in batches") with an ON-CHIP event scheduler: every block keeps a pool of P particles in shared memory
// (structure of arrays) and loops over four phases, each of which runs one kind of work on a COMPACTED index list,
// so that all 32 lanes of a warp execute the same event type:
//   R  refill   free slots take fission children from the global ring queue, then new source histories (A.3, A.6)
//   F  flight   distances, event choice, track-length score, move (A.2, A.4, A.7); census bookkeeping (A.8)
//   S  surface  boundary condition / neighbour cell (A.5)
//   C  collide  reaction choice, scattering or fission (A.6); a fission parent continues as its first child,
//               the other children go to the global queue
// Lists are built with ballot-aggregated shared-memory atomics.  Particle records never travel through HBM; only
// the fission queue, the batch accumulators (fp64 RED) and the counters do.  Trajectories depend on
// (seed, history id, lineage) alone, so the order in which the lists are processed is free.
#pragma once
#include "mcdc_kernels.cuh"

namespace mcdc {

struct PoolCtl {                   // block-wide control words (shared memory)
  uint32_t nF[2], nS, nC, nFree;
  uint32_t got, n_src, src_base, nfree_old;
  unsigned long long qbase;
  int done, src_done;
  double led[LED_N];               // block ledger: production capture fission_abs leak census_final lost
  unsigned long long n_coll, n_surf, n_census, n_children, n_lost, n_src_total, n_src_lost;
};

// ballot-aggregated append to a shared-memory list; returns this lane's index (valid when want)
__device__ __forceinline__ uint32_t list_append(uint32_t *counter, bool want) {
  const unsigned m = __ballot_sync(MCDC_FULL, want);
  if (m == 0u) return 0u;
  const int leader = __ffs(m) - 1;
  uint32_t base = 0u;
  if (lane_id() == leader) base = atomicAdd(counter, (uint32_t)__popc(m));
  base = __shfl_sync(MCDC_FULL, base, leader);
  return base + (uint32_t)__popc(m & ((1u << lane_id()) - 1u));
}

// warp total of v added to *dst by one lane (skipped when every lane holds zero)
__device__ __forceinline__ void warp_accumulate(double *dst, double v) {
  if (__ballot_sync(MCDC_FULL, v != 0.0) == 0u) return;
  v = warp_sum(v);
  if (lane_id() == 0) atomicAdd(dst, v);
}
__device__ __forceinline__ void warp_accumulate_u(unsigned long long *dst, uint32_t v) {
  if (__ballot_sync(MCDC_FULL, v != 0u) == 0u) return;
  v = __reduce_add_sync(MCDC_FULL, v);
  if (lane_id() == 0) atomicAdd(dst, (unsigned long long)v);
}

__host__ __device__ inline size_t pool_bytes_per_slot() { return 8 * 8 + 8 + 8 * 4 + 2 + 5 * 2; }   // 116

template <bool STAGED, bool FAST, int NT>
__global__ void __launch_bounds__(NT, 1) k_pool(Tables T, HistoryArgs A) {
  __shared__ PoolCtl ctl;
  const TB<STAGED> tb(T);
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const uint32_t P = A.pool_slots;
  // ---- carve the dynamic shared memory: [staged tables][census populations][pool arrays][lists] ----
  unsigned char *base = g_smem + A.smem_tables;
  double *s_popw = reinterpret_cast<double *>(base); base += (size_t)T.K * 8;
  uint32_t *s_popn = reinterpret_cast<uint32_t *>(base); base += ((size_t)T.K * 4 + 15) / 16 * 16;
  double *px = reinterpret_cast<double *>(base), *py = px + P, *pz = py + P, *pux = pz + P, *puy = pux + P, *puz = puy + P,
         *pt = puz + P, *pw = pt + P;
  unsigned long long *pkey = reinterpret_cast<unsigned long long *>(pw + P);
  uint32_t *pctr = reinterpret_cast<uint32_t *>(pkey + P), *phid = pctr + P;
  int *pcell = reinterpret_cast<int *>(phid + P), *pg = pcell + P, *plast = pg + P, *ppk = plast + P, *pit = ppk + P,
      *pev = pit + P;
  uint16_t *pslot = reinterpret_cast<uint16_t *>(pev + P);
  uint16_t *LF0 = pslot + P, *LF1 = LF0 + P, *LS = LF1 + P, *LC = LS + P, *LFREE = LC + P;

  if (STAGED) {
    const uint4 *src = reinterpret_cast<const uint4 *>(T.blob);
    uint4 *dst = reinterpret_cast<uint4 *>(g_smem);
    for (uint32_t i = tid; i < T.hot_bytes / 16u; i += NT) dst[i] = src[i];
  }
  for (int k = tid; k < T.K; k += NT) { s_popw[k] = 0.0; s_popn[k] = 0u; }
  for (uint32_t i = tid; i < P; i += NT) LFREE[i] = (uint16_t)(P - 1u - i);
  if (tid == 0) {
    ctl.nF[0] = ctl.nF[1] = ctl.nS = ctl.nC = 0u; ctl.nFree = P;
    ctl.got = ctl.n_src = ctl.src_base = ctl.nfree_old = 0u; ctl.qbase = 0ull; ctl.done = 0; ctl.src_done = 0;
    for (int e = 0; e < LED_N; ++e) ctl.led[e] = 0.0;
    ctl.n_coll = ctl.n_surf = ctl.n_census = ctl.n_children = ctl.n_lost = ctl.n_src_total = ctl.n_src_lost = 0ull;
  }
  __syncthreads();
  unsigned long long *q_head = A.q.head_tail, *q_tail = A.q.head_tail + 1;
  const unsigned long long q_cap = (unsigned long long)A.q.mask + 1ull;
  uint32_t *ev_rec = A.ev;
  int par = 0;

  for (;;) {
    // =============== R: acquire work for the free slots (one thread), then initialise the new particles ===============
    if (tid == 0) {
      ctl.nS = 0u; ctl.nC = 0u;
      const uint32_t nfree = ctl.nFree;
      uint32_t got = 0u, n_src = 0u, src_base = 0u;
      unsigned long long qbase = 0ull;
      int done = *(volatile int *)&A.cnt->overflow;      // a queue overflow was flagged somewhere: the run is void
      if (!done && nfree > 0u) {
        const unsigned long long h = ld_volatile_u64(q_head), t = ld_volatile_u64(q_tail);
        if (t > h) {
          const unsigned long long want = min((unsigned long long)nfree, t - h);
          if (atomicCAS(q_head, h, h + want) == h) { got = (uint32_t)want; qbase = h; }
        }
        if (!ctl.src_done && nfree > got) {
          const uint32_t want = nfree - got;
          src_base = atomicAdd(A.hist_cursor, want);
          if (src_base >= A.n_hist) { n_src = 0u; ctl.src_done = 1; }
          else {
            n_src = min(want, A.n_hist - src_base);
            if (src_base + want >= A.n_hist) ctl.src_done = 1;
          }
        }
        if (got == 0u && n_src == 0u && nfree == P && ctl.src_done) {
          const unsigned long long h2 = ld_volatile_u64(q_head), t2 = ld_volatile_u64(q_tail);
          if (t2 <= h2) done = 1;                         // pool empty, no source left, queue empty
        }
      }
      ctl.got = got; ctl.qbase = qbase; ctl.n_src = n_src; ctl.src_base = src_base; ctl.nfree_old = nfree;
      ctl.nFree = nfree - got - n_src;
      ctl.done = done;
      ctl.n_src_total += n_src;
    }
    __syncthreads();                                                                          // barrier 1
    if (ctl.done) break;
    uint16_t *Fcur = par ? LF1 : LF0, *Fnxt = par ? LF0 : LF1;
    uint32_t *nFcur = &ctl.nF[par], *nFnxt = &ctl.nF[par ^ 1];
    bool give_back = false;
    uint32_t give_slot = 0u;
    {
      const uint32_t got = ctl.got, total = ctl.got + ctl.n_src, nfree_old = ctl.nfree_old;
      double lost_w = 0.0;
      uint32_t lost_n = 0u;
      for (uint32_t b = (uint32_t)wid * 32u; b < total; b += NT) {
        const uint32_t li = b + lane;
        const bool act = li < total;
        bool ok = act;
        uint32_t i = 0u;
        if (act) {
          i = LFREE[nfree_old - 1u - li];
          PState p;
          int pk, it, kind;
          if (li < got) {                                  // a fission child from the global queue (A.6)
            const unsigned long long qi = ctl.qbase + li;
            const uint32_t j = (uint32_t)qi & A.q.mask;
            const uint32_t expect = (uint32_t)(qi + 1ull);
            for (uint32_t spin = 0; ld_acquire_u32(A.q.flag + j) != expect; ++spin) {
              if ((spin & 255u) == 255u && (*(volatile int *)&A.cnt->overflow || spin > (1u << 26))) {
                atomicExch(&A.cnt->overflow, 1);           // producer gave up (overflow) or never published
                ok = false;
                break;
              }
            }
            p.x = A.q.x[j]; p.y = A.q.y[j]; p.z = A.q.z[j]; p.t = A.q.t[j]; p.w = A.q.w[j];
            p.key = A.q.key[j];
            const int4 m = A.q.meta[j];
            p.cell = m.x; pk = m.y; p.hid = (uint32_t)m.z; it = m.w;
            p.ctr = 0u;
            kind = FI_CHILD;
          } else {                                         // a new source history (A.3)
            p.hid = ctl.src_base + (li - got);
            source_position(T, A.seed_mixed, A.first_history + p.hid, p);
            pk = census_index(tb, p.t);
            it = 0;
            kind = FI_SOURCE;
          }
          p.g = 0;
          if (ok && !flight_init(tb, p, kind)) { ok = false; lost_w += p.w; lost_n += 1u; }   // source outside every cell
          if (ok) {
            px[i] = p.x; py[i] = p.y; pz[i] = p.z; pux[i] = p.ux; puy[i] = p.uy; puz[i] = p.uz; pt[i] = p.t; pw[i] = p.w;
            pkey[i] = p.key; pctr[i] = p.ctr; phid[i] = p.hid; pcell[i] = p.cell; pg[i] = p.g; plast[i] = -1;
            ppk[i] = pk; pit[i] = it; pslot[i] = (uint16_t)(p.hid / A.hb);
          } else { give_back = true; give_slot = i; }
        }
        const uint32_t at = list_append(nFcur, ok);
        if (ok) Fcur[at] = (uint16_t)i;
      }
      warp_accumulate(&ctl.led[LED_LOST], lost_w);
      warp_accumulate_u(&ctl.n_src_lost, lost_n);
    }
    __syncthreads();                                                                          // barrier 2
    if (__ballot_sync(MCDC_FULL, give_back) != 0u) {       // rare: slots of particles that could not start
      const uint32_t at = list_append(&ctl.nFree, give_back);
      if (give_back) LFREE[at] = (uint16_t)give_slot;
    }

    // =============== F: flight -- distances, event choice, score, move (A.2, A.4, A.7, A.8) ===============
    {
      const uint32_t nf = *nFcur;
      double led_final = 0.0;
      uint32_t n_census = 0u;
      for (uint32_t b = (uint32_t)wid * 32u; b < nf; b += NT) {
        const uint32_t li = b + lane;
        const bool act = li < nf;
        const uint32_t i = act ? Fcur[li] : 0u;
        PState p;
        int pk = 0, it = 0;
        if (act) {
          p.x = px[i]; p.y = py[i]; p.z = pz[i]; p.ux = pux[i]; p.uy = puy[i]; p.uz = puz[i]; p.t = pt[i]; p.w = pw[i];
          p.key = pkey[i]; p.ctr = pctr[i]; p.cell = pcell[i]; p.g = pg[i]; p.last_surf = plast[i];
          pk = ppk[i]; it = pit[i];
        } else {
          p.x = p.y = p.z = p.ux = p.uy = p.t = p.w = 0.0; p.uz = 1.0;
          p.key = 0ull; p.ctr = 0u; p.cell = 0; p.g = 0; p.last_surf = -1;
        }
        p.hid = 0u;
        p.ix = 1.0 / p.ux; p.iy = 1.0 / p.uy; p.iz = 1.0 / p.uz;
        double d = 0.0, pos_star = 0.0;
        int ev = -1, slot_star = -1, which = -1;
        const double t_census = tb.census(pk);
        if (act) ev = find_event_typed(tb, p, t_census, d, slot_star, which, pos_star);
        {
          TallySink S;
          S.slab = nullptr; S.global_x = A.x_acc + (size_t)pslot[i] * T.n_bins; S.slab_lo = 0; S.slab_bins = 0;
          S.aggregate = A.aggregate;
          if (FAST) score_track_fast(tb, S, act, p, it, d);
          else score_track(tb, S, act, p.x, p.y, p.z, p.ux, p.uy, p.uz, p.t, p.w, p.g, d);
        }
        int census_k = -1;
        bool to_F = false, dead = false;
        if (act) {
          px[i] = p.x + d * p.ux; py[i] = p.y + d * p.uy; pz[i] = p.z + d * p.uz;
          pt[i] = (ev == EV_CENSUS) ? t_census : p.t + d * tb.inv_speed(p.g);
          pctr[i] = p.ctr; pit[i] = it;
          if (ev == EV_CENSUS) {                           // A.8: bookkeeping only, then the next interval
            census_k = pk;
            n_census += 1u;
            if (d > 0.0) plast[i] = -1;
            if (pk == T.K - 1) { led_final += p.w; dead = true; }
            else { ppk[i] = pk + 1; to_F = true; }
            if (ev_rec) atomicAdd(ev_rec + (size_t)phid[i] * 4 + 3, 1u);
          } else if (ev == EV_SURFACE) {
            pev[i] = slot_star | (which << 28);
          }
        }
        // census population, merged inside the warp
        if (__ballot_sync(MCDC_FULL, census_k >= 0) != 0u) {
          double v = p.w;
          const bool absorbed = warp_merge_equal<int>(census_k, census_k >= 0, v, 4);
          if (census_k >= 0) {
            if (!absorbed) atomicAdd(s_popw + census_k, v);
            atomicAdd(s_popn + census_k, 1u);
          }
        }
        uint32_t at = list_append(nFnxt, to_F);
        if (to_F) Fnxt[at] = (uint16_t)i;
        at = list_append(&ctl.nS, ev == EV_SURFACE);
        if (ev == EV_SURFACE) LS[at] = (uint16_t)i;
        at = list_append(&ctl.nC, ev == EV_COLLISION);
        if (ev == EV_COLLISION) LC[at] = (uint16_t)i;
        at = list_append(&ctl.nFree, dead);
        if (dead) LFREE[at] = (uint16_t)i;
      }
      warp_accumulate(&ctl.led[LED_CENSUS_FINAL], led_final);
      warp_accumulate_u(&ctl.n_census, n_census);
    }
    __syncthreads();                                                                          // barrier 3
    if (tid == 0) { ctl.n_surf += ctl.nS; ctl.n_coll += ctl.nC; *nFcur = 0u; }

    // =============== S: surface events (A.5) ===============
    {
      const uint32_t ns = ctl.nS;
      double led_leak = 0.0, led_lost = 0.0;
      uint32_t n_lost = 0u;
      for (uint32_t b = (uint32_t)wid * 32u; b < ns; b += NT) {
        const uint32_t li = b + lane;
        const bool act = li < ns;
        const uint32_t i = act ? LS[li] : 0u;
        bool alive = false;
        if (act) {
          PState p;
          p.x = px[i]; p.y = py[i]; p.z = pz[i]; p.ux = pux[i]; p.uy = puy[i]; p.uz = puz[i]; p.w = pw[i];
          p.ix = p.iy = p.iz = 0.0;
          p.cell = pcell[i]; p.last_surf = -1;
          const int e = pev[i];
          const int slot_star = e & 0x0FFFFFFF, which = (e >> 28) & 7;
          const int cell0 = p.cell;
          const double ux0 = p.ux, uy0 = p.uy, uz0 = p.uz;
          double pos_star = 0.0;
          if (which < 6) pos_star = tb.template ldb<double>(T.o_cell_rec + (uint32_t)p.cell * CELL_REC_BYTES + CR_BOUND + 8u * which);
          alive = surface_event_typed(tb, p, slot_star, which, pos_star, &led_leak, &led_lost, &n_lost);
          plast[i] = p.last_surf;
          if (alive) {
            if (p.cell != cell0) pcell[i] = p.cell;
            if (p.ux != ux0) pux[i] = p.ux;
            if (p.uy != uy0) puy[i] = p.uy;
            if (p.uz != uz0) puz[i] = p.uz;
          }
          if (ev_rec) atomicAdd(ev_rec + (size_t)phid[i] * 4 + 1, 1u);
        }
        uint32_t at = list_append(nFnxt, alive);
        if (alive) Fnxt[at] = (uint16_t)i;
        at = list_append(&ctl.nFree, act && !alive);
        if (act && !alive) LFREE[at] = (uint16_t)i;
      }
      warp_accumulate(&ctl.led[LED_LEAK], led_leak);
      warp_accumulate(&ctl.led[LED_LOST], led_lost);
      warp_accumulate_u(&ctl.n_lost, n_lost);
    }

    // =============== C: collisions (A.6) ===============
    {
      const uint32_t nc = ctl.nC;
      double led_cap = 0.0, led_fis = 0.0, led_prod = 0.0;
      uint32_t n_children = 0u;
      for (uint32_t b = (uint32_t)wid * 32u; b < nc; b += NT) {
        const uint32_t li = b + lane;
        const bool act = li < nc;
        const uint32_t i = act ? LC[li] : 0u;
        PState p;
        p.key = pkey[i]; p.ctr = pctr[i]; p.cell = pcell[i]; p.g = pg[i]; p.w = pw[i];
        p.x = p.y = p.z = p.t = 0.0; p.ux = p.uy = 0.0; p.uz = 1.0; p.hid = 0u; p.last_surf = -1;
        int fi = FI_NONE, n_push = 0;
        uint32_t c0 = 0u;
        bool alive = false;
        if (act) {
          const int r = collision_event(tb, p, c0, &led_cap, &led_fis, &led_prod);
          if (r == -1) { fi = FI_SCATTER; alive = true; }
          else if (r > 0) { n_children += (uint32_t)r; n_push = r - 1; alive = true; }
          if (ev_rec) {
            atomicAdd(ev_rec + (size_t)phid[i] * 4 + 0, 1u);
            if (r > 0) atomicAdd(ev_rec + (size_t)phid[i] * 4 + 2, (uint32_t)r);
          }
        }
        // fission: publish children 1..n-1 to the global queue, continue as child 0
        if (__ballot_sync(MCDC_FULL, n_push > 0) != 0u) {
          int pre = n_push;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(MCDC_FULL, pre, o);
            if (lane >= o) pre += v;
          }
          const int total = __shfl_sync(MCDC_FULL, pre, 31);
          unsigned long long qb = 0ull;
          int okq = 1;
          if (lane == 0) {
            qb = atomicAdd(q_tail, (unsigned long long)total);
            if (qb + (unsigned long long)total - ld_volatile_u64(q_head) + 65536ull > q_cap) okq = 0;
          }
          qb = __shfl_sync(MCDC_FULL, qb, 0) + (unsigned long long)(pre - n_push);
          okq = __shfl_sync(MCDC_FULL, okq, 0);
          if (!okq && lane == 0) atomicExch(&A.cnt->overflow, 1);
          if (n_push > 0 && okq) {
            const double x = px[i], y = py[i], z = pz[i], t = pt[i];
            const int4 meta = make_int4(p.cell, ppk[i], (int)phid[i], pit[i]);
            for (int c = 0; c < n_push; ++c) {
              const uint32_t j = (uint32_t)(qb + (unsigned long long)c) & A.q.mask;
              A.q.x[j] = x; A.q.y[j] = y; A.q.z[j] = z; A.q.t[j] = t; A.q.w[j] = p.w;
              A.q.key[j] = child_key(p.key, c0, (uint32_t)(c + 1));
              A.q.meta[j] = meta;
            }
            __threadfence();
            for (int c = 0; c < n_push; ++c) {
              const unsigned long long qi = qb + (unsigned long long)c;
              st_release_u32(A.q.flag + ((uint32_t)qi & A.q.mask), (uint32_t)(qi + 1ull));
            }
          }
        }
        if (alive && fi == FI_NONE) {                      // fission parent -> its first child, in place
          p.key = child_key(p.key, c0, 0u);
          p.ctr = 0u;
          fi = FI_CHILD;
          pkey[i] = p.key;
        }
        if (alive) {
          flight_init(tb, p, fi);                          // group and direction of the outgoing flight
          pg[i] = p.g; pux[i] = p.ux; puy[i] = p.uy; puz[i] = p.uz; pctr[i] = p.ctr;
        }
        if (act) plast[i] = -1;
        uint32_t at = list_append(nFnxt, alive);
        if (alive) Fnxt[at] = (uint16_t)i;
        at = list_append(&ctl.nFree, act && !alive);
        if (act && !alive) LFREE[at] = (uint16_t)i;
      }
      warp_accumulate(&ctl.led[LED_CAPTURE], led_cap);
      warp_accumulate(&ctl.led[LED_FISSION_ABS], led_fis);
      warp_accumulate(&ctl.led[LED_PRODUCTION], led_prod);
      warp_accumulate_u(&ctl.n_children, n_children);
    }
    __syncthreads();                                                                          // barrier 4
    par ^= 1;
  }

  // ---- block totals ----
  __syncthreads();
  for (int k = tid; k < T.K; k += NT) {
    if (s_popn[k] != 0u) { atomicAdd(A.pop_w + k, s_popw[k]); atomicAdd(A.pop_n + k, (unsigned long long)s_popn[k]); }
  }
  if (tid == 0) {
    DevCounters *cnt = A.cnt;
    for (int e = 0; e < LED_N; ++e)
      if (ctl.led[e] != 0.0) atomicAdd(&cnt->ledger[1 + e], ctl.led[e]);
    atomicAdd(&cnt->ledger[0], (double)ctl.n_src_total);
    atomicAdd(&cnt->n[0], ctl.n_src_total);
    atomicAdd(&cnt->n[1], ctl.n_coll + ctl.n_surf + ctl.n_census);
    atomicAdd(&cnt->n[2], ctl.n_coll);
    atomicAdd(&cnt->n[3], ctl.n_surf);
    atomicAdd(&cnt->n[4], ctl.n_census);
    atomicAdd(&cnt->n[5], ctl.n_children);
    atomicAdd(&cnt->n[6], ctl.n_lost + ctl.n_src_lost);
  }
}

}  // namespace mcdc
