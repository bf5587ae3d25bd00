// phs_kernels.cu -- CTA path of the hot path in CUDA for sm_100a: activation, max-min progressive filling (fair
// share per link, bottleneck argmin, freeze/scatter), event advance, retire + DAG release.
// a4-a9.  One CTA simulates one instance start to finish with ALL dynamic state in shared memory.
//
// Algorithm.  The paper's water-filling freezes ONE bottleneck link per iteration (PAPER.md
// L165).  Because rates live on an exact integer grid (reading R-FX), freezing EVERY link whose (share, id) key is
// smaller than the key of every link it shares an unfrozen flow with ("local minimum") in one parallel round gives
// bit-identical rates and bottleneck ids (proof in DESIGN.md).  A link is a local minimum iff no unfrozen flow on
// it names another link as the arg-min of its own path: every flow stamps the links it does NOT vote for with the
// round's number ("beaten"), and freezes if its own arg-min link carries no stamp of this round.  No counters, no
// atomics, nothing to clear.
// Rates are a function of the active set of a static link component only, and (reading R-LZ) a flow's state
// changes only when its own rate changes, so an event re-solves just the components it touched.
// Phases of one event (barrier-separated):
//   X   flows whose completion time equals t_next retire and release their successors; slots whose activation
//       time has come become ACTIVE (a8, a4); both stamp their component "to solve"
//   V0  every flow of a stamped component refreshes the fair share of its links (a5), picks its arg-min (a6)
//   F0  flows whose arg-min link is unbeaten freeze at its share (a7); a changed rate settles the flow's
//       remaining bytes and gives a new completion time; all threads fold the slot times into the next t_next (a8)
//   I/D/V/F  only when flows are left: working capacities are set up, frozen flows debit their paths, and the
//       rounds repeat on the debited shares
#include <cuda_runtime.h>

#include <climits>
#include <cstdio>

#include "phs_device.h"
#include "phs_devutil.cuh"

namespace phs {

namespace {

// ------------------------------------------------------------------------------------------------ smem layout
struct CtaSmem {
  // per link [L]
  long long *l_cap, *l_share0, *l_caprem, *l_sharew;
  int *l_n0;      // ACTIVE flows on the link
  int *l_chg;     // solve id of the last change of l_n0 (share0 is stale for that solve until recomputed)
  int *l_beat;    // round number in which some unfrozen flow on the link voted for another link
  int *l_nw;      // working: unfrozen flows on the link (rounds >= 1)
  int *l_deb;     // working: round number of the last debit
  int *l_solve;   // per component (indexed by its representative link): id of the solve that must redo it
  int *l_won;     // LOG: round in which the link froze flows (counts bottleneck links once)
  int *l_gid;     // link id of the topology (the links of a unit are numbered densely)
  unsigned *l_rmin;  // INC, per component (representative link): limit below which rates stand in this event's solve
  // per slot [S]: one slot per PENDING or ACTIVE flow
  double *s_tc;   // PENDING: activation time; ACTIVE: completion time; free: +inf
  double *s_rem;  // remaining bytes at time s_tl
  double *s_tl;   // time of the last rate change
  long long *s_rq;  // rate in quanta, -1 before the first solve
  int4 *s_meta;   // .x flow id (-1 = free); .y -2 PENDING, -1 ACTIVE and unfrozen, >= 0 bottleneck link;
                  // .z static link component; .w arg-min link of the current round
  uint4 *s_path;  // the path as 8 x uint16 (kNoLink = none): one 16-byte load brings the whole path
  int *s_succ_cnt, *s_succ0, *s_succ1;
  int *free_q;    // FIFO ring of free slots
  unsigned *pc8;  // [(PCF+7)/8] predecessor counters, 4 bits per flow
  double *red;    // [32] per-warp partial minima
  long long *red_key;  // [32] LOG: per-warp partial first_bneck key
  int *red_id;    // [32]
  int *ctl;       // [32] control words
};
enum {
  C_HI = 0, C_QHEAD, C_QTAIL, C_NACTIVE, C_NPEND, C_OVERFLOW, C_DONE, C_EV_NCOMP, C_EV_ROUNDS, C_EV_NACT0,
  C_EV_NACT1, C_ADDED, C_NCTL
};

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

constexpr unsigned kNoLink = 0xffffu;
constexpr int kRminShift = 30;  // rates are below 2^62 quanta: rate >> 30 is one 32-bit word (a more careful limit)
static_assert(kMaxHops <= 8, "a path is stored as 8 x uint16");
// unpack link h of a packed path
__device__ __forceinline__ int path_at(const uint4 &p, int h) {
  const unsigned w = h < 2 ? p.x : h < 4 ? p.y : h < 6 ? p.z : p.w;
  return (int)((h & 1) ? (w >> 16) : (w & 0xffffu));
}

// `lean` (CtaLaunch::lean): bit 0 = the arrays only a solve with a second round touches (l_caprem, l_sharew, l_nw,
// l_deb) and the link ids (l_gid, read once per completion) are not in shared memory -- the kernel points them at a
// per-CTA global scratch region and at the unit's linkid table; bit 1 = l_cap likewise reads the unit's capq table.
// With `lean` the carved pointers of those fields are not valid.
__host__ __device__ inline size_t carve(CtaSmem *s, unsigned char *base, int L, int S, int pcf, bool log, int lean) {
  size_t o = 0, a;
#define PHS_TAKE(field, type, count)                    \
  a = o;                                                \
  o = align_up(o + sizeof(type) * (size_t)(count), 16); \
  if (s) s->field = (type *)(base + a);
  const int Lw = (lean & 1) ? 0 : L, Lcap = (lean & 2) ? 0 : L;
  PHS_TAKE(l_cap, long long, Lcap)
  PHS_TAKE(l_share0, long long, L)
  PHS_TAKE(l_caprem, long long, Lw)
  PHS_TAKE(l_sharew, long long, Lw)
  PHS_TAKE(s_tc, double, S)
  PHS_TAKE(s_rem, double, S)
  PHS_TAKE(s_tl, double, S)
  PHS_TAKE(s_rq, long long, S)
  PHS_TAKE(red, double, 32)
  PHS_TAKE(red_key, long long, log ? 32 : 0)
  PHS_TAKE(l_n0, int, L)
  PHS_TAKE(l_chg, int, L)
  PHS_TAKE(l_beat, int, L)
  PHS_TAKE(l_nw, int, Lw)
  PHS_TAKE(l_deb, int, Lw)
  PHS_TAKE(l_solve, int, L)
  PHS_TAKE(l_won, int, log ? L : 0)
  PHS_TAKE(l_gid, int, Lw)
  PHS_TAKE(l_rmin, unsigned, (lean & 4) ? L : 0)  // bit 2: incremental re-solve (never together with bits 0 / 1)
  PHS_TAKE(s_meta, int4, S)
  PHS_TAKE(s_path, uint4, S)
  PHS_TAKE(s_succ_cnt, int, S)
  PHS_TAKE(s_succ0, int, S)
  PHS_TAKE(s_succ1, int, S)
  PHS_TAKE(free_q, int, S)
  PHS_TAKE(pc8, unsigned, (pcf + 7) / 8)
  PHS_TAKE(red_id, int, log ? 32 : 0)
  PHS_TAKE(ctl, int, 32)
#undef PHS_TAKE
  return o;
}

// 64-bit add on a shared-memory word with two native 32-bit atomics (a 64-bit atomicAdd on shared memory compiles
// to a compare-and-swap loop).  Exact once all adds of a phase have completed: every carry out of the low word is
// added to the high word exactly once.
__device__ __forceinline__ void smem_add64(long long *p, long long v) {
  unsigned *w = (unsigned *)p;
  const unsigned lo = (unsigned)(unsigned long long)v, hi = (unsigned)((unsigned long long)v >> 32);
  const unsigned old = atomicAdd(w, lo);
  const unsigned carry = (old + lo) < old ? 1u : 0u;
  if (hi + carry) atomicAdd(w + 1, hi + carry);
}

// min over the warp of non-negative doubles (their bit patterns order like unsigned integers): two REDUX steps
__device__ __forceinline__ double warp_min_nonneg(double v) {
  const unsigned long long b = (unsigned long long)__double_as_longlong(v);
  const unsigned hi = (unsigned)(b >> 32), lo = (unsigned)b;
  const unsigned mhi = __reduce_min_sync(0xffffffffu, hi);
  const unsigned mlo = __reduce_min_sync(0xffffffffu, hi == mhi ? lo : 0xffffffffu);
  return __longlong_as_double((long long)(((unsigned long long)mhi << 32) | mlo));
}

}  // namespace

size_t cta_smem_bytes(int n_links, int slots, int pc_flows, bool log, int lean) {
  return carve(nullptr, nullptr, n_links, slots, pc_flows, log, lean);
}
size_t cta_lean_scratch_bytes(int n_links) {  // per CTA: l_caprem, l_sharew (8 each), l_nw, l_deb (4 each)
  return align_up((size_t)n_links * 24, 256);
}

// ================================================================================================ CTA kernel
// NT threads; LOG: write the event log (and solve every component at every event, so that the log's iteration
// count and first bottleneck are those of a from-scratch solve); PCS: predecessor counters live in shared memory;
// HIST: record the throughput history (a call in the hottest block of the kernel: compiled out when not wanted).
// INC: incremental re-solve (the rule of phs_cluster.cu / phs_grid.cu): for units whose solves take
// several filling rounds (all-to-all, raw flow sets).  l_caprem then persists from solve to solve, an event re-solves
// only the flows at or above its limit; ring traffic (one round per solve) is better off without it.
template <int NT, bool LOG, bool PCS, bool HIST, bool INC = false>
__global__ void __launch_bounds__(NT, (NT <= 128 ? 1024 : 512) / NT) phs_cta_kernel(DevTables T, const int32_t *__restrict__ order, int n_order,
                                                     int *ticket, int SC, int pcf, int lean,
                                                     unsigned char *lean_scratch) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int sh_inst;
  CtaSmem S;
  const int L = T.n_links;
  const size_t smem_used = carve(&S, smem_raw, L, SC, pcf, LOG, lean);
  if (lean & 1) {  // working arrays of multi-round solves: this CTA's region of the global scratch (L2-resident)
    unsigned char *w = lean_scratch + (size_t)blockIdx.x * align_up((size_t)L * 24, 256);
    S.l_caprem = (long long *)w;
    S.l_sharew = S.l_caprem + L;
    S.l_nw = (int *)(S.l_sharew + L);
    S.l_deb = S.l_nw + L;
  }
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NW = NT / 32;

  for (;;) {
    // ---- a9: dynamic instance queue
    if (tid == 0) sh_inst = atomicAdd(ticket, 1);
    __syncthreads();
    const int qi = sh_inst;
    __syncthreads();
    if (qi >= n_order) break;
    const int inst = order[qi];
    const InstDesc D = T.inst[inst];
    const FlowRec *__restrict__ rec = T.rec + D.flow_base;
    const int32_t *__restrict__ succ = T.succ + D.succ_base;
    int32_t *pred_cnt = T.pred_cnt + D.flow_base;
    const uint32_t *__restrict__ fmap = T.fmap + D.flow_base;  // unit-local flow -> position in the outputs
    double *t_done = T.t_done;
    int32_t *bneck_out = T.bneck;
    const int64_t *__restrict__ capq = T.capq + D.link_base;
    const int32_t *__restrict__ linkid = T.linkid + D.link_base;
    const int Li = D.n_links;  // <= L, the launch-wide maximum the shared-memory layout is carved for
    phs_event *log = (LOG && D.log_base >= 0) ? T.log + D.log_base : nullptr;
    const int F = D.n_flows;

    // phs_run_until: a unit that stopped at an earlier t_stop continues from its parked state
    const bool resuming =
        T.resume && T.park && ((const ParkRegs *)(T.park + (size_t)inst * T.park_stride))->valid;
    // ---- init: nothing active, every slot free
    // lean layout: capacities and link ids are read where they are (the unit's tables)
    const long long *l_cap = (lean & 2) ? (const long long *)capq : S.l_cap;
    const int *l_gid = (lean & 1) ? (const int *)linkid : S.l_gid;
    if (!resuming)
    for (int l = tid; l < Li; l += NT) {
      if (!(lean & 2)) S.l_cap[l] = capq[l];
      if (!(lean & 1)) S.l_gid[l] = linkid[l];
      S.l_n0[l] = 0;
      S.l_chg[l] = 0;
      S.l_beat[l] = 0;
      S.l_deb[l] = 0;
      S.l_solve[l] = 0;
      if (LOG) S.l_won[l] = 0;
      if (INC) {
        S.l_caprem[l] = capq[l];
        S.l_nw[l] = 0;
        S.l_rmin[l] = 0xffffffffu;
      }
    }
    // the scratch region served another unit (or another CTA parked this one): no debit stamp may look current.
    // No solve is in progress between events, and round numbers compared with l_deb are >= 1.
    if (resuming && (lean & 1))
      for (int l = tid; l < Li; l += NT) S.l_deb[l] = 0;
    if (!resuming) {
    for (int s = tid; s < SC; s += NT) {
      S.s_meta[s].x = -1;
      S.s_tc[s] = kInf;
    }
    if (tid < C_NCTL) S.ctl[tid] = 0;
    }
    if (PCS && !resuming) {
      const unsigned *src = (const unsigned *)(T.pred_cnt0_u8 + D.pc8_base);
      for (int w = tid; w < (F + 7) / 8; w += NT) S.pc8[w] = src[w];
    }
    __syncthreads();

    // one slot per flow that is PENDING or ACTIVE; the whole record is staged when the flow becomes PENDING
    auto fill_slot = [&](int slot, int out, const FlowRec &r, double ta) {
      S.s_meta[slot].x = out;  // where the flow's results go; its unit-local id is not needed any more
      S.s_rem[slot] = r.bytes;
      S.s_meta[slot].y = -2;
      S.s_meta[slot].z = r.comp;
      {
        unsigned w[4] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0xffffffffu};
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {
          const unsigned l = r.path[h] < 0 ? kNoLink : (unsigned)r.path[h];
          w[h >> 1] = (h & 1) ? ((w[h >> 1] & 0xffffu) | (l << 16)) : ((w[h >> 1] & 0xffff0000u) | l);
        }
        S.s_path[slot] = make_uint4(w[0], w[1], w[2], w[3]);
      }
      S.s_succ_cnt[slot] = r.succ_cnt;
      S.s_succ0[slot] = r.succ_in[0];
      S.s_succ1[slot] = r.succ_in[1];
      S.s_tc[slot] = ta;
    };

    // S4: flows without predecessors become PENDING at t_act = start + Lat
    if (!resuming) {
      const int32_t *__restrict__ pc0 = T.pred_cnt0 + D.flow_base;
      for (int f = tid; f < F; f += NT) {
        int pc;
        if (PCS) {
          pc = (S.pc8[f >> 3] >> ((f & 7) * 4)) & 0xf;
        } else {
          pc = pc0[f];
          pred_cnt[f] = pc;
        }
        if (pc == 0) {
          const FlowRec r = rec[f];
          const int slot = atomicAdd(&S.ctl[C_HI], 1);
          if (slot < SC) {
            fill_slot(slot, (int)fmap[f], r, __dadd_rn(r.start, r.lat));
            atomicAdd(&S.ctl[C_NPEND], 1);
          } else {
            S.ctl[C_OVERFLOW] = 1;
          }
        }
      }
    }
    __syncthreads();

    double now = 0.0, t_next = 0.0;
    int ev = -1;      // index of the event whose advance phase X is about to execute
    int solve = 0;    // id of the solve that follows the current phase X
    int g = 0;        // filling-round number, unique over the instance
    long long sum_active = 0, sum_rounds = 0;
    int max_active = 0, max_pending = 0;
    int status = PHS_OK;
    int first_bneck = -1;
    if (resuming) {  // shared memory and the loop-carried registers as they were when the unit stopped
      const ParkRegs *park = (const ParkRegs *)(T.park + (size_t)inst * T.park_stride);
      const uint4 *src = (const uint4 *)((const unsigned char *)park + sizeof(ParkRegs));
      uint4 *dst = (uint4 *)smem_raw;
      for (size_t i = tid; i < smem_used / 16; i += NT) dst[i] = src[i];
      now = park->now;
      t_next = park->t_next;
      sum_active = park->sum_active;
      sum_rounds = park->sum_rounds;
      ev = park->ev;
      solve = park->solve;
      g = park->g;
      max_active = park->max_active;
      max_pending = park->max_pending;
      first_bneck = park->first_bneck;
      __syncthreads();
    }
#ifdef PHS_PHASE_CLOCKS
    long long pc_[8] = {0, 0, 0, 0, 0, 0, 0, 0}, pt_ = clock64();
// BAR.SYNC does not block at issue: read a barrier-protected word before taking the clock
#define PHS_TICK(i) { if (*(volatile int *)&S.ctl[C_HI] < -5) pt_ = 0; const long long t_ = clock64(); pc_[i] += t_ - pt_; pt_ = t_; }
#else
#define PHS_TICK(i)
#endif

    // Snapshot of the slot high-water mark and of the free queue's tail as phase X of the next event must see them.
    // Taken where a barrier protects it (here, and right after the X barrier of every event): nothing changes the two
    // words between an X barrier and the next phase X, while a read at the top of phase X would race with the atomics
    // of warps that are already inside it.
    int hi_carry = min(S.ctl[C_HI], SC), qtail_carry = S.ctl[C_QTAIL];

    for (;;) {
      if (t_next > T.t_stop) {  // phs_run_until: the next event lies beyond the requested time
        status = kPaused;
        break;
      }
      // ======== phase X (a8 + a4): retire what completes at t_next, release successors, activate what is due
      ++solve;
      const int hi0 = hi_carry;
      const int qtail = qtail_carry;

      auto activate = [&](int slot) {  // PENDING -> ACTIVE: the flow now counts on its links
        const uint4 pv = S.s_path[slot];
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {
          const int l = path_at(pv, h);
          if (l != (int)kNoLink) {
            atomicAdd(&S.l_n0[l], 1);
            S.l_chg[l] = solve;
          }
        }
        S.l_solve[S.s_meta[slot].z] = solve;
        if (INC) S.ctl[C_ADDED] = 1;  // its links bound what stands (pass A)
        S.s_rq[slot] = -1;
        S.s_meta[slot].y = -1;
        S.s_tc[slot] = kInf;
        atomicAdd(&S.ctl[C_NACTIVE], 1);
        atomicSub(&S.ctl[C_NPEND], 1);
        if (LOG) atomicAdd(&S.ctl[C_EV_NACT0 + ((ev + 1) & 1)], 1);
        // the successors' records will be needed when this flow completes: pull them towards L2 now
        const int nsucc = S.s_succ_cnt[slot];
        if (nsucc > 0 && nsucc <= 2) {
          asm volatile("prefetch.global.L1 [%0];" ::"l"(rec + S.s_succ0[slot]));
          if (nsucc > 1) asm volatile("prefetch.global.L1 [%0];" ::"l"(rec + S.s_succ1[slot]));
        }
      };
      auto pred_done = [&](int gf) {  // S4.5: pred_cnt--; true when it reaches 0
        if (PCS) {
          const unsigned sh = (unsigned)(gf & 7) * 4u;  // a counter is >= 1 here, so the subtraction never borrows
          const unsigned old = atomicSub(&S.pc8[gf >> 3], 1u << sh);
          return ((old >> sh) & 0xfu) == 1u;
        }
        return atomicSub(&pred_cnt[gf], 1) == 1;
      };
      // -> PENDING with t_act = max(start, now) + Lat.  `reuse` >= 0: the slot the releasing flow just vacated (no
      // trip through the free queue); it is consumed by the first successor that needs a slot.
      auto make_pending = [&](int out, const FlowRec &r, int &reuse) {
        const double ta = __dadd_rn(r.start > t_next ? r.start : t_next, r.lat);
        int slot = reuse;
        reuse = -1;
        if (slot < 0) {
          const int h = atomicAdd(&S.ctl[C_QHEAD], 1);
          slot = h < qtail ? S.free_q[h % SC] : atomicAdd(&S.ctl[C_HI], 1);
        }
        if (slot >= SC) {
          S.ctl[C_OVERFLOW] = 1;
          return;
        }
        atomicAdd(&S.ctl[C_NPEND], 1);
        const bool due = ta <= t_next;  // zero path latency: due at this very timestamp
        fill_slot(slot, out, r, due ? kInf : ta);
        if (due) activate(slot);
      };
      auto release2 = [&](int g0, int g1, int &reuse) {  // both counters, then both records: the loads overlap
        const bool z0 = g0 >= 0 && pred_done(g0);
        const bool z1 = g1 >= 0 && pred_done(g1);
        FlowRec r0, r1;
        int o0 = 0, o1 = 0;
        if (z0) {
          r0 = rec[g0];
          o0 = (int)fmap[g0];
        }
        if (z1) {
          r1 = rec[g1];
          o1 = (int)fmap[g1];
        }
        if (z0) make_pending(o0, r0, reuse);
        if (z1) make_pending(o1, r1, reuse);
      };

      for (int s = tid; s < hi0; s += NT) {
        if (!(S.s_tc[s] <= t_next)) continue;  // free slots hold +inf
        if (S.s_meta[s].y == -2) {
          activate(s);
          continue;
        }
        // the flow completes at t_next (bit-equal absolute time, S4.4)
        const int f = S.s_meta[s].x;
        t_done[f] = t_next;
        bneck_out[f] = l_gid[S.s_meta[s].y];
        const uint4 pv = S.s_path[s];
        const long long rq_done = INC ? S.s_rq[s] : 0;
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {
          const int l = path_at(pv, h);
          if (l != (int)kNoLink) {
            atomicSub(&S.l_n0[l], 1);
            S.l_chg[l] = solve;
            if (INC) smem_add64(&S.l_caprem[l], rq_done);  // the flow's rate goes back to its links
          }
        }
        S.l_solve[S.s_meta[s].z] = solve;
        if (INC) atomicMin(&S.l_rmin[S.s_meta[s].z], (unsigned)(rq_done >> kRminShift));
        const int nsucc = S.s_succ_cnt[s], sc0 = S.s_succ0[s], sc1 = S.s_succ1[s];
        S.s_meta[s].x = -1;
        S.s_tc[s] = kInf;
        atomicSub(&S.ctl[C_NACTIVE], 1);
        atomicAdd(&S.ctl[C_DONE], 1);
        if (LOG) atomicAdd(&S.ctl[C_EV_NCOMP], 1);
        int reuse = s;  // the vacated slot goes to the first successor that becomes PENDING, else to the free queue
        if (nsucc <= 2) {
          if (nsucc > 0) release2(sc0, nsucc > 1 ? sc1 : -1, reuse);
        } else {
          for (int e = 0; e < nsucc; ++e) release2(succ[sc0 + e], -1, reuse);
        }
        if (reuse >= 0) S.free_q[atomicAdd(&S.ctl[C_QTAIL], 1) % SC] = s;
      }
      PHS_TICK(0)
      __syncthreads();
      PHS_TICK(1)
      now = t_next;
      if (tid == 0) {
        if (S.ctl[C_QHEAD] > qtail) S.ctl[C_QHEAD] = qtail;  // pops that found the queue empty took fresh slots
        if (LOG) {
          if (log && ev >= 0) {  // O4: the event that just finished
            phs_event e;
            e.t = now;
            e.n_completed = S.ctl[C_EV_NCOMP];
            e.n_activated = S.ctl[C_EV_NACT0 + (ev & 1)];
            e.n_rounds = S.ctl[C_EV_ROUNDS];
            e.first_bneck = first_bneck;
            log[ev] = e;
          }
          S.ctl[C_EV_NCOMP] = 0;
          S.ctl[C_EV_ROUNDS] = 0;
          if (ev >= 0) S.ctl[C_EV_NACT0 + (ev & 1)] = 0;
        }
      }
      ++ev;
      if (S.ctl[C_OVERFLOW]) {
        status = kOverflow;
        break;
      }
      const int nA = S.ctl[C_NACTIVE];
      const int nPend = S.ctl[C_NPEND];
      if (nA == 0 && nPend == 0) break;  // S4.3: nothing active, nothing pending -> stop
      const int hi = hi_carry = min(S.ctl[C_HI], SC);
      qtail_carry = S.ctl[C_QTAIL];
      max_active = max(max_active, nA);
      max_pending = max(max_pending, nPend);

      const int added = INC ? S.ctl[C_ADDED] : 0;  // (reset after the next barrier, below)
      // ======== a5: fair share of the links whose flow count changed in this event, one thread per link
      if (!INC) {
        for (int l = tid; l < Li; l += NT) {
          if (S.l_chg[l] != solve) continue;
          const int n = S.l_n0[l];
          if (n > 0) S.l_share0[l] = fair_share(l_cap[l], n);
        }
        __syncthreads();
      }

      // ======== rates (a6-a7): parallel progressive filling over the components this event touched
      auto in_solve = [&](int s) {  // ACTIVE flow of a component that must be re-solved
        const int4 m = S.s_meta[s];
        if (m.x < 0 || m.y == -2) return false;
        return LOG || S.l_solve[m.z] == solve;
      };
      auto freeze = [&](int s, int arg, long long rq) {  // a7; R-LZ: only a changed rate touches the flow's state
        S.s_meta[s].y = arg;
        const long long old = S.s_rq[s];
        if (rq != old) {
          double rem = S.s_rem[s];
          if (old >= 0) {  // settle at the old rate: mul, sub, clamp
            rem = __dsub_rn(rem, __dmul_rn(rate_of(old), __dsub_rn(now, S.s_tl[s])));
            rem = rem > 0.0 ? rem : 0.0;
            S.s_rem[s] = rem;
          }
          S.s_tl[s] = now;
          S.s_rq[s] = rq;
          if (HIST) append_history(T.hist, T.hist_n, T.hist_cap, now, rq, (uint32_t)S.s_meta[s].x, (uint32_t)ev);
          S.s_tc[s] = __dadd_rn(now, __ddiv_rn(rem, rate_of(rq)));  // S4.3: division, then addition
        }
        if (LOG && atomicExch(&S.l_won[arg], g) != g) atomicAdd(&S.ctl[C_EV_ROUNDS], 1);
      };
      int rounds = 1;
      if (INC) {
        if (added) {
          // ---- A: flows were ADDED.  A link that carries an added flow keeps a share of at least floor(cap / n) -- n its
          // flow count now -- all through the new solve: every flow slower than the smallest such share stands.
          for (int s = tid; s < hi; s += NT) {
            const int4 m = S.s_meta[s];
            if (m.x < 0 || m.y != -1 || S.s_rq[s] >= 0) continue;  // ACTIVE and never solved = added
            const uint4 pv = S.s_path[s];
            long long mn = LLONG_MAX;
#pragma unroll
            for (int h = 0; h < kMaxHops; ++h) {
              const int l = path_at(pv, h);
              if (l == (int)kNoLink) continue;
              const long long sh = fair_share(l_cap[l], S.l_n0[l]);
              mn = sh < mn ? sh : mn;
            }
            atomicMin(&S.l_rmin[m.z], (unsigned)(mn >> kRminShift));
          }
          __syncthreads();
        }
        // ---- C: the flows at or above their component's limit give their rates back to their links and count as
        // unfrozen again; stamp l_deb = g makes the first vote below compute the links' shares from (caprem, nw)
        ++g;
        for (int s = tid; s < hi; s += NT) {
          const int4 m = S.s_meta[s];
          if (m.x < 0 || m.y == -2 || S.l_solve[m.z] != solve) continue;
          const long long rq = S.s_rq[s];
          if (rq >= 0 && (unsigned)(rq >> kRminShift) < S.l_rmin[m.z]) continue;  // below the limit: stands
          S.s_meta[s].y = -1;
          const uint4 pv = S.s_path[s];
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {
            const int l = path_at(pv, h);
            if (l == (int)kNoLink) continue;
            if (rq > 0) smem_add64(&S.l_caprem[l], rq);
            atomicAdd(&S.l_nw[l], 1);
            S.l_deb[l] = g;
          }
        }
      }
      if (!INC) ++g;
      if (!INC) {  // ---- V0: fair share of the links whose flow count changed (a5), arg-min link of every flow (a6)
        long long bk = LLONG_MAX;
        int bl = INT_MAX;
        for (int s = tid; s < hi; s += NT) {
          if (!in_solve(s)) continue;
          S.s_meta[s].y = -1;
          const uint4 pv = S.s_path[s];
          int p[kMaxHops];
          long long sh[kMaxHops];
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {  // all loads first
            p[h] = path_at(pv, h);
            sh[h] = S.l_share0[p[h] != (int)kNoLink ? p[h] : 0];
          }
          long long best = LLONG_MAX;
          int arg = -1;
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {
            const int l = p[h];
            if (l == (int)kNoLink) continue;
            if (sh[h] < best || (sh[h] == best && l < arg)) {
              best = sh[h];
              arg = l;
            }
          }
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h)
            if (p[h] != (int)kNoLink && p[h] != arg) S.l_beat[p[h]] = g;  // an unfrozen flow on p[h] prefers another link
          S.s_meta[s].w = arg;
          if (LOG && (best < bk || (best == bk && arg < bl))) {
            bk = best;
            bl = arg;
          }
        }
        if (LOG) {  // O4 first_bneck = global arg-min = min over the flows' arg-mins
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) {
            const long long ok = __shfl_xor_sync(0xffffffffu, bk, o);
            const int ol = __shfl_xor_sync(0xffffffffu, bl, o);
            if (ok < bk || (ok == bk && ol < bl)) {
              bk = ok;
              bl = ol;
            }
          }
          if (lane == 0) {
            S.red_key[warp] = bk;
            S.red_id[warp] = bl;
          }
        }
      }
      PHS_TICK(2)
      __syncthreads();
      PHS_TICK(3)
      bool left = INC;  // INC: the rounds below do all the solving (and fold the slot times even if nothing is unfrozen)
      if (INC) {        // every thread has read the limits and the flag: ready for the next event
        for (int l = tid; l < Li; l += NT)
          if (S.l_solve[l] == solve) S.l_rmin[l] = 0xffffffffu;
        if (tid == 0) S.ctl[C_ADDED] = 0;
      }
      if (!INC) {  // ---- F0: unbeaten arg-min links freeze their flows (a7); fold the slot times (a8)
        double mymin = kInf;
        for (int s = tid; s < hi; s += NT) {
          if (S.s_meta[s].x < 0) continue;
          if (S.s_meta[s].y == -1) {
            const int arg = S.s_meta[s].w;
            if (S.l_beat[arg] != g)
              freeze(s, arg, S.l_share0[arg]);
            else
              left = true;
          }
          mymin = dmin(mymin, S.s_tc[s]);
        }
        const double wm = warp_min_nonneg(mymin);
        if (lane == 0) S.red[warp] = wm;
      }
      PHS_TICK(4)
      left = __syncthreads_or(left);
      PHS_TICK(5)
      if (left) {
        if (!INC) {
        // ---- I: working capacities of the links of this solve (idempotent stores)
        for (int s = tid; s < hi; s += NT) {
          if (!in_solve(s)) continue;
          const uint4 pv = S.s_path[s];
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {
            const int l = path_at(pv, h);
            if (l == (int)kNoLink) continue;
            S.l_caprem[l] = l_cap[l];
            S.l_nw[l] = S.l_n0[l];
            S.l_sharew[l] = S.l_share0[l];
          }
        }
        __syncthreads();
        // ---- D: flows frozen in the first round debit their paths (a7)
        for (int s = tid; s < hi; s += NT) {
          if (!in_solve(s) || S.s_meta[s].y < 0) continue;
          const long long rq = S.s_rq[s];
          const uint4 pv = S.s_path[s];
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {
            const int l = path_at(pv, h);
            if (l == (int)kNoLink) continue;
            if (S.l_n0[l] > 1) {
              smem_add64(&S.l_caprem[l], -rq);
              atomicSub(&S.l_nw[l], 1);
              S.l_deb[l] = g;
            }
          }
        }
        __syncthreads();
        }
        for (;;) {
          ++g;
          ++rounds;
          // ---- V: shares of the links debited in the previous round, arg-min of every unfrozen flow
          for (int s = tid; s < hi; s += NT) {
            if (S.s_meta[s].x < 0 || S.s_meta[s].y != -1) continue;
            const uint4 pv = S.s_path[s];
            int p[kMaxHops];
            long long best = LLONG_MAX;
            int arg = -1;
#pragma unroll
            for (int h = 0; h < kMaxHops; ++h) {
              const int l = p[h] = path_at(pv, h);
              if (l == (int)kNoLink) continue;
              long long sh;
              if (S.l_deb[l] == g - 1) {
                sh = fair_share(S.l_caprem[l], S.l_nw[l]);
                S.l_sharew[l] = sh;
              } else {
                sh = S.l_sharew[l];
              }
              if (sh < best || (sh == best && l < arg)) {
                best = sh;
                arg = l;
              }
            }
#pragma unroll
            for (int h = 0; h < kMaxHops; ++h)
              if (p[h] != (int)kNoLink && p[h] != arg) S.l_beat[p[h]] = g;
            S.s_meta[s].w = arg;
          }
          __syncthreads();
          // ---- F: freeze, debit, fold
          left = false;
          double mymin = kInf;
          for (int s = tid; s < hi; s += NT) {
            if (S.s_meta[s].x < 0) continue;
            if (S.s_meta[s].y == -1) {
              const int arg = S.s_meta[s].w;
              if (S.l_beat[arg] != g) {
                const long long rq = S.l_sharew[arg];
                freeze(s, arg, rq);
                const uint4 pv = S.s_path[s];
#pragma unroll
                for (int h = 0; h < kMaxHops; ++h) {
                  const int l = path_at(pv, h);
                  if (l == (int)kNoLink) continue;
                  if (INC || S.l_n0[l] > 1) {  // INC: caprem persists, so every freeze is booked
                    smem_add64(&S.l_caprem[l], -rq);
                    atomicSub(&S.l_nw[l], 1);
                    S.l_deb[l] = g;
                  }
                }
              } else {
                left = true;
              }
            }
            mymin = dmin(mymin, S.s_tc[s]);
          }
          const double wm = warp_min_nonneg(mymin);
          if (lane == 0) S.red[warp] = wm;
          left = __syncthreads_or(left);
          if (!left) break;
        }
      }
      // ======== next time (a8): t_next = min over completion times and pending activation times
      t_next = S.red[0];
#pragma unroll
      for (int w = 1; w < NW; ++w) t_next = dmin(t_next, S.red[w]);
      if (LOG && tid == 0) {
        first_bneck = -1;
        if (nA > 0) {
          long long bk = S.red_key[0];
          first_bneck = S.red_id[0];
          for (int w = 1; w < NW; ++w)
            if (S.red_key[w] < bk || (S.red_key[w] == bk && S.red_id[w] < first_bneck)) {
              bk = S.red_key[w];
              first_bneck = S.red_id[w];
            }
        }
      }
      sum_active += nA;
      sum_rounds += rounds;
      PHS_TICK(6)
    }
    if (T.park) {  // park the unit if it stopped at t_stop; a finished unit has nothing to resume
      ParkRegs *park = (ParkRegs *)(T.park + (size_t)inst * T.park_stride);
      if (status == kPaused) {
        __syncthreads();
        uint4 *dst = (uint4 *)((unsigned char *)park + sizeof(ParkRegs));
        const uint4 *src = (const uint4 *)smem_raw;
        for (size_t i = tid; i < smem_used / 16; i += NT) dst[i] = src[i];
      }
      if (tid == 0) {
        ParkRegs r;
        r.now = now; r.t_next = t_next; r.sum_active = sum_active; r.sum_rounds = sum_rounds;
        r.ev = ev; r.solve = solve; r.g = g; r.max_active = max_active; r.max_pending = max_pending;
        r.first_bneck = first_bneck; r.valid = status == kPaused ? 1 : 0; r.n_windows = 0;
        *park = r;
      }
    }
#ifdef PHS_PHASE_CLOCKS
    if ((tid == 0 || tid == NT - 1) && F > 3000 && inst < 40)
      printf("inst %d tid %d events %d cycles: X %lld waitX %lld V0 %lld wait1 %lld F0 %lld wait2 %lld rest %lld\n", inst, tid,
             ev, pc_[0], pc_[1], pc_[2], pc_[3], pc_[4], pc_[5], pc_[6]);
#endif
    if (tid == 0) {
      if (status == PHS_OK && S.ctl[C_DONE] < F) status = PHS_ECYCLE;  // WAITING flows left over
      InstResult r;
      r.status = status;
      r.path = 0;
      r.n_events = ev;
      r.sum_active = sum_active;
      r.sum_par_rounds = sum_rounds;
      r.max_active = max_active;
      r.max_pending = max_pending;
      r.max_slots = S.ctl[C_HI];
      r.n_windows = ev;  // one event per iteration on this path
      T.res[inst] = r;
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------ launchers
namespace {
template <int NT, bool LOG, bool PCS, bool HIST>
cudaError_t launch_hist(const DevTables &t, const int32_t *order, int n, int *ticket, const CtaLaunch &c,
                        cudaStream_t stream) {
  cudaError_t e = cudaFuncSetAttribute(phs_cta_kernel<NT, LOG, PCS, HIST>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
  if (e != cudaSuccess) return e;
  phs_cta_kernel<NT, LOG, PCS, HIST><<<c.grid, NT, c.smem, stream>>>(t, order, n, ticket, c.slots, c.pc_flows, c.lean,
                                                                    c.lean_scratch);
  return cudaGetLastError();
}
template <int NT, bool PCS>
cudaError_t launch_inc(const DevTables &t, const int32_t *order, int n, int *ticket, const CtaLaunch &c,
                       cudaStream_t stream) {  // incremental re-solve: no event log, no history
  cudaError_t e = cudaFuncSetAttribute(phs_cta_kernel<NT, false, PCS, false, true>,
                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);
  if (e != cudaSuccess) return e;
  phs_cta_kernel<NT, false, PCS, false, true><<<c.grid, NT, c.smem, stream>>>(t, order, n, ticket, c.slots, c.pc_flows,
                                                                             c.lean, c.lean_scratch);
  return cudaGetLastError();
}
template <int NT, bool LOG, bool PCS>
cudaError_t launch_one(const DevTables &t, const int32_t *order, int n, int *ticket, const CtaLaunch &c,
                       cudaStream_t stream) {
  return t.hist ? launch_hist<NT, LOG, PCS, true>(t, order, n, ticket, c, stream)
                : launch_hist<NT, LOG, PCS, false>(t, order, n, ticket, c, stream);
}
template <int NT>
cudaError_t launch_nt(const DevTables &t, const int32_t *order, int n, int *ticket, const CtaLaunch &c,
                      cudaStream_t stream) {
  const bool pcs = c.pc_flows > 0;
  if ((c.lean & 4) && !c.log && !t.hist)
    return pcs ? launch_inc<NT, true>(t, order, n, ticket, c, stream) : launch_inc<NT, false>(t, order, n, ticket, c, stream);
  if (c.log) return pcs ? launch_one<NT, true, true>(t, order, n, ticket, c, stream)
                        : launch_one<NT, true, false>(t, order, n, ticket, c, stream);
  return pcs ? launch_one<NT, false, true>(t, order, n, ticket, c, stream)
             : launch_one<NT, false, false>(t, order, n, ticket, c, stream);
}
}  // namespace

cudaError_t launch_cta_path(const DevTables &t, const int32_t *order, int n, int *ticket, const CtaLaunch &c,
                            cudaStream_t stream) {
  switch (c.threads) {
    case 32:
      return launch_nt<32>(t, order, n, ticket, c, stream);
    case 64:
      return launch_nt<64>(t, order, n, ticket, c, stream);
    case 128:
      return launch_nt<128>(t, order, n, ticket, c, stream);
    case 256:
      return launch_nt<256>(t, order, n, ticket, c, stream);
    case 512:
      return launch_nt<512>(t, order, n, ticket, c, stream);
    default:
      return cudaErrorInvalidValue;
  }
}

// ------------------------------------------------------------------------------------------------ a10: results
// O5: per-collective finish time = max t_done over its (contiguous) flows; one warp per collective.
__global__ void phs_collective_times_kernel(const double *__restrict__ t_done, const int64_t *__restrict__ first,
                                            const int32_t *__restrict__ nflows, int64_t n_colls,
                                            double *__restrict__ out) {
  const int64_t c = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (c >= n_colls) return;
  const double *p = t_done + first[c];
  const int n = nflows[c];
  double m = 0.0;
  bool open_flows = false;  // after phs_run_until: a collective with unfinished flows (NaN) has no finish time yet
  for (int i = lane; i < n; i += 32) {
    open_flows |= p[i] != p[i];
    m = fmax(m, p[i]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  open_flows = __any_sync(0xffffffffu, open_flows);
  if (lane == 0) out[c] = open_flows ? __longlong_as_double(0x7ff8000000000000LL) : m;
}

// NEXT-1: results later than t are forgotten (completion time NaN, bottleneck -1), as after a stop at time t
__global__ void phs_forget_after_kernel(double *__restrict__ t_done, int32_t *__restrict__ bneck, int64_t n, double t) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n && !(t_done[i] <= t)) {
    t_done[i] = __longlong_as_double(-1LL);  // the all-ones pattern cudaMemset(0xff) leaves: a NaN
    bneck[i] = -1;
  }
}

cudaError_t launch_forget_after(double *t_done, int32_t *bneck, int64_t n, double t, cudaStream_t stream) {
  if (n == 0) return cudaSuccess;
  phs_forget_after_kernel<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(t_done, bneck, n, t);
  return cudaGetLastError();
}

cudaError_t launch_collective_times(const double *t_done, const int64_t *coll_first, const int32_t *coll_nflows,
                                    int64_t n_colls, double *out, cudaStream_t stream) {
  if (n_colls == 0) return cudaSuccess;
  const int threads = 256;
  const int64_t blocks = (n_colls * 32 + threads - 1) / threads;
  phs_collective_times_kernel<<<(unsigned)blocks, threads, 0, stream>>>(t_done, coll_first, coll_nflows, n_colls, out);
  return cudaGetLastError();
}

}  // namespace phs
