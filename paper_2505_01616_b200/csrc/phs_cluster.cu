// phs_cluster.cu -- cluster path of the hot path: one thread-block cluster (up to 16 CTAs, hardware cluster
// barrier) simulates one LARGE instance (SURVEY.md 8(a) a4-a9 for instances whose state does not fit one SM).
// Same algorithm as the CTA path (phs_kernels.cu): stamp-based local-minimum test, static-component re-solve, lazy
// settle (R-LZ).  ALL dynamic state stays on chip, spread over the shared memory of the cluster's CTAs:
//   * link l is owned by CTA (l mod CS); its 64 bytes of state sit in the owner's shared memory and every CTA
//     reads / stamps / debits them through distributed shared memory (DSMEM, ~200 cycles instead of an L2 trip);
//   * each CTA owns a private set of flow slots in its own shared memory (a flow is created in the CTA that
//     released it); cold slot fields spill to a CTA-private global partition only when shared memory is short;
//   * per-CTA partial results (next-event time, flows-left flag, flow counts) are written to arrays in CTA 0's
//     shared memory and read back by everybody after the barrier;
//   * per filling round: V (shares, arg-min, beat stamps) | cluster barrier | F (freeze, settle, debit) | cluster
//     barrier.  No value-returning global atomic and no L2 round trip sits on the per-round path.
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include <climits>
#include <cstdio>

#include "phs_device.h"
#include "phs_devutil.cuh"

namespace cg = cooperative_groups;

namespace phs {

namespace {

constexpr int NT = kClusterThreads;
constexpr unsigned short kNoLink = 0xffff;
constexpr int kMaxCS = 16;
constexpr int kRminShift = 30;  // capacities are below 2^42 byte/s = 2^62 quanta (phs_set_link_capacities): 32 bits left

struct LinkA {  // 32 bytes: what a flow reads when it votes in the first round
  long long share0;  // floor(cap / n0), valid unless chg == current solve id
  long long cap;
  int n0;     // ACTIVE flows on the link
  int chg;    // solve id of the last change of n0
  int beat;   // round number in which an unfrozen flow on the link voted for another link
  int solve;  // (indexed by a component's representative link) id of the solve that must redo the component
};
struct LinkB {  // 32 bytes: working state of a solve's debits
  long long caprem;
  long long sharew;  // share after debits, valid iff wsolve == current solve id
  int nw;            // unfrozen flows on the link
  int deb;           // round number of the last debit
  int wsolve;
  int comp;          // static component (representative link) of the link
};

// per-CTA partial results, gathered in CTA 0's shared memory
struct CombX {  // after phase X
  int n_act, n_pend, n_done, over;
  int hi, ev_ncomp, ev_nact, pad;
};
struct CombF {  // after a filling round
  double tmin;
  long long fb_key;
  int fb_id, left, pad0, pad1;
};
struct Comb {
  CombX x[kMaxCS];
  CombF f[kMaxCS];
  int ev_rounds;
  int inst;
};

struct Slots {
  double *tc;          // PENDING: activation time; ACTIVE: completion time; free: +inf
  long long *rq;       // rate in quanta, -1 before the first solve
  int *bn;             // -3 free, -2 PENDING, -1 ACTIVE and unfrozen, >= 0 bottleneck link
  unsigned short *comp, *arg;
  unsigned short *path;  // [Sc * kMaxHops]
  unsigned short *wl0, *wl1;
  // cold fields: shared memory when it fits, else global
  double *rem, *tl;
  int *flow, *succ_cnt, *succ0, *succ1, *freeq;
};
constexpr int kSlotHotBytes = 8 + 8 + 4 + 2 * 2 + 2 * kMaxHops + 2 * 2;  // 40
constexpr int kSlotColdBytes = 2 * 8 + 5 * 4;                            // 36

__host__ __device__ inline size_t up16(size_t x) { return (x + 15) / 16 * 16; }

// dynamic shared memory of one CTA
__host__ __device__ inline size_t smem_layout(int L, int CS, int64_t Sc, bool agg, bool cold_smem, bool log, bool repl,
                                              size_t *o_lb, size_t *o_won, size_t *o_beatf, size_t *o_agg,
                                              size_t *o_repl, size_t *o_hot, size_t *o_cold) {
  const size_t Lc = (size_t)(L + CS - 1) / CS;
  size_t o = 0;
  o += Lc * sizeof(LinkA);
  if (o_lb) *o_lb = o;
  o += Lc * sizeof(LinkB);
  if (o_won) *o_won = o;
  o += up16(log ? Lc * 4 : 0);
  if (o_beatf) *o_beatf = o;
  o += 2 * up16((size_t)L * 4);  // beatf[L], csolve[L]
  if (o_agg) *o_agg = o;
  o += agg ? up16((size_t)L * 16) : 0;
  if (o_repl) *o_repl = o;
  // sh_loc[L], sh0_loc[L] (8 each), chg_loc[L] (4), comp_loc[L] (2); with pre-aggregation and without the log (incremental
  // re-solve) also crmin[L] (4)
  o += repl ? up16(up16((size_t)L * 22) + ((agg && !log) ? (size_t)L * 4 : 0)) : 0;
  if (o_hot) *o_hot = o;
  o += up16((size_t)Sc * kSlotHotBytes);
  if (o_cold) *o_cold = o;
  o += cold_smem ? up16((size_t)Sc * kSlotColdBytes) : 0;
  return o;
}

__device__ __forceinline__ void add64_2x32(long long *p, long long v) {  // works on local and remote smem
  unsigned *w = (unsigned *)p;
  const unsigned lo = (unsigned)(unsigned long long)v, hi = (unsigned)((unsigned long long)v >> 32);
  const unsigned old = atomicAdd(w, lo);
  const unsigned carry = (old + lo) < old ? 1u : 0u;
  if (hi + carry) atomicAdd(w + 1, hi + carry);
}

enum { M_HI = 0, M_QHEAD, M_QTAIL, M_NACT, M_NPEND, M_NDONE, M_NWL0, M_NWL1, M_NTOUCH, M_OVER, M_EVC, M_EVA, M_ADDED,
       M_NCTL };

}  // namespace

size_t cluster_smem_bytes(int L, int cluster_size, int64_t Sc, bool aggregate, bool cold_smem, bool log,
                          bool replicate) {
  return smem_layout(L, cluster_size, Sc, aggregate, cold_smem, log, replicate, nullptr, nullptr, nullptr, nullptr,
                     nullptr, nullptr, nullptr);
}
size_t cluster_park_cta_bytes(int L, int cluster_size, int64_t Sc, bool aggregate, bool cold_smem, bool log,
                              bool replicate) {
  const size_t b = cluster_smem_bytes(L, cluster_size, Sc, aggregate, cold_smem, log, replicate) + 64 + sizeof(Comb) +
                   (cold_smem ? 0 : (size_t)Sc * kSlotColdBytes + 16);  // + 16: the copies move whole 16-byte words
  return (b + 255) / 256 * 256;
}
size_t cluster_region_bytes(int64_t Sc, int cluster_size) {  // global spill area of the cold slot fields
  return (size_t)cluster_size * (((size_t)Sc * kSlotColdBytes + 255) / 256 * 256);
}

// ================================================================================================ cluster kernel
// LOG: write the event log (and solve every component at every event); AGG: a CTA first sums its debits per link
// in its own shared memory and then debits each touched link once.
template <bool LOG, bool AGG>
__global__ void __launch_bounds__(kClusterThreads, 1)
    phs_cluster_kernel(DevTables T, const int32_t *__restrict__ list, int n_list, int *ticket, ClusterScratch SC) {
  cg::cluster_group cluster = cg::this_cluster();
  const int CS = (int)cluster.num_blocks();
  const int crank = (int)cluster.block_rank();
  const int csh = 31 - __clz(CS), cmask = CS - 1;  // CS is a power of two
  const int region = blockIdx.x / CS;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int ctid = crank * NT + tid;
  const int CT = CS * NT;
  const int L = T.n_links;
  const int Lc = (L + CS - 1) / CS;
  const int Sc = (int)SC.Sc;

  extern __shared__ __align__(16) unsigned char smem_raw[];
  size_t o_lb, o_won, o_beatf, o_agg, o_repl, o_hot, o_cold;
  const bool REPL = SC.replicate != 0;
  const size_t smem_used = smem_layout(L, CS, Sc, AGG, SC.cold_smem != 0, LOG, REPL, &o_lb, &o_won, &o_beatf, &o_agg,
                                       &o_repl, &o_hot, &o_cold);
  // REPL: every CTA keeps its own copy of the links' current fair shares, so that voting reads local shared
  // memory; owners broadcast the shares they recompute after debits, stale first-round shares are refreshed by the
  // flows that need them
  // INC, incremental re-solve: an event leaves untouched every flow whose rate is below the smallest
  // rate among the flows it REMOVES -- the one-bottleneck-per-iteration algorithm freezes links in ascending (share, id)
  // order, and its iterations before a removed flow's own bottleneck do not see the removal -- and below the smallest
  // floor(cap / n) over the links of the flows it ADDS (such a link's share never falls below that in the new solve).
  // Per component, crmin = the smaller of the two limits; the capacity left on every link after ALL frozen flows
  // (caprem) persists from solve to solve, and the flows at or above the limit credit their rates back.
  const bool INCS = REPL && AGG && !LOG;            // the layout has crmin[]
  const bool INC = INCS && SC.incremental != 0;
  long long *sh_loc = (long long *)(smem_raw + o_repl);  // [L] share in the current round
  long long *sh0_loc = sh_loc + L;                        // [L] share at the start of a solve
  int *chg_loc = (int *)(sh0_loc + L);                    // [L] solve id of the last change of the link's flow count
  unsigned short *comp_loc = (unsigned short *)(chg_loc + L);  // [L] static component of every link
  // [L] per component (representative link), replicated per CTA: the smallest removed rate of the event, truncated to
  // rate >> kRminShift so that it is one 32-bit word (a remote 32-bit min needs no answer; truncation only makes the cut
  // more careful: (rate >> k) < (r_min >> k) implies rate < r_min)
  unsigned *crmin = INCS ? (unsigned *)(smem_raw + o_repl + up16((size_t)L * 22)) : nullptr;
  LinkA *la = (LinkA *)smem_raw;
  LinkB *lb = (LinkB *)(smem_raw + o_lb);
  int *won = (int *)(smem_raw + o_won);
  int *beatf = (int *)(smem_raw + o_beatf);
  int *csolve = beatf + (up16((size_t)L * 4) / 4);  // per component (representative link): solve id that must redo it;
                                                    // replicated in every CTA, because every flow and link reads it
  long long *dcap_loc = (long long *)(smem_raw + o_agg);
  int *dn_loc = (int *)(dcap_loc + L);
  int *touched = dn_loc + L;
  Slots S;
  {
    unsigned char *h = smem_raw + o_hot;
    S.tc = (double *)h;
    S.rq = (long long *)(S.tc + Sc);
    S.bn = (int *)(S.rq + Sc);
    S.comp = (unsigned short *)(S.bn + Sc);
    S.arg = S.comp + Sc;
    S.path = S.arg + Sc;
    S.wl0 = S.path + (size_t)Sc * kMaxHops;
    S.wl1 = S.wl0 + Sc;
    unsigned char *c = SC.cold_smem ? smem_raw + o_cold
                                    : SC.base + (size_t)region * SC.region_bytes +
                                          (size_t)crank * (((size_t)Sc * kSlotColdBytes + 255) / 256 * 256);
    S.rem = (double *)c;
    S.tl = S.rem + Sc;
    S.flow = (int *)(S.tl + Sc);
    S.succ_cnt = S.flow + Sc;
    S.succ0 = S.succ_cnt + Sc;
    S.succ1 = S.succ0 + Sc;
    S.freeq = S.succ1 + Sc;
  }
  __shared__ Comb comb;  // x / f.tmin / f.left: every CTA has the cluster's values; the rest: CTA 0's copy is used
  __shared__ double red[32];
  __shared__ long long red_key[32];
  __shared__ int red_id[32];
  __shared__ int ctl[M_NCTL];
  __shared__ int bc[10];      // broadcast of the cluster-wide counts to the CTA
  __shared__ double bc_t;     // ... and of the next event time
  Comb *comb0 = cluster.map_shared_rank(&comb, 0);

  // state of link l lives in the shared memory of CTA (l mod CS)
  auto LA = [&](int l) { return cluster.map_shared_rank(la + (l >> csh), (unsigned)(l & cmask)); };
  auto LB = [&](int l) { return cluster.map_shared_rank(lb + (l >> csh), (unsigned)(l & cmask)); };

  for (;;) {
    // ---- a9: clusters pull instances from the list
    if (ctid == 0) comb.inst = atomicAdd(ticket, 1);
    cluster.sync();
    const int qi = comb0->inst;
    cluster.sync();
    if (qi >= n_list) break;
    const int inst = list[qi];
    const InstDesc D = T.inst[inst];
    const FlowRec *__restrict__ rec = T.rec + D.flow_base;
    const int32_t *__restrict__ succ = T.succ + D.succ_base;
    const int32_t *__restrict__ pc0 = T.pred_cnt0 + D.flow_base;
    int32_t *pred_cnt = T.pred_cnt + D.flow_base;
    const uint32_t *__restrict__ fmap = T.fmap + D.flow_base;  // unit-local flow -> position in the outputs
    double *t_done = T.t_done;
    int32_t *bneck_out = T.bneck;
    const int64_t *__restrict__ capq = T.capq + D.link_base;
    const int32_t *__restrict__ lcomp = T.lcomp + D.link_base;
    const int32_t *__restrict__ linkid = T.linkid + D.link_base;
    const int Li = D.n_links;  // <= L, the launch-wide maximum the shared-memory layout is sized for
    phs_event *log = (LOG && D.log_base >= 0) ? T.log + D.log_base : nullptr;
    const int F = D.n_flows;

    // phs_run_until: a unit that stopped at an earlier t_stop continues from its parked state
    const int pidx = SC.park ? SC.park_index[inst] : -1;
    unsigned char *upark = pidx >= 0 ? SC.park + (size_t)pidx * SC.park_unit_stride : nullptr;
    unsigned char *cpark = upark ? upark + kClusterParkHeader + (size_t)crank * SC.park_cta_stride : nullptr;
    const bool resuming = SC.resume && upark && ((const ClusterParkRegs *)upark)->valid;  // the same in every CTA
    // ---- init: own links, own slots
    if (!resuming) {
    for (int li = tid; li < Lc; li += NT) {
      const int l = li * CS + crank;
      LinkA a;
      a.share0 = 0; a.cap = l < Li ? capq[l] : 0; a.n0 = 0; a.chg = 0; a.beat = 0; a.solve = 0;
      la[li] = a;
      LinkB b;
      b.caprem = INC ? a.cap : 0; b.sharew = 0; b.nw = 0; b.deb = 0; b.wsolve = 0; b.comp = l < Li ? lcomp[l] : 0;
      lb[li] = b;
      if (LOG) won[li] = 0;
    }
    for (int l = tid; l < L; l += NT) {
      beatf[l] = 0;
      csolve[l] = 0;
      if (INCS) crmin[l] = 0xffffffffu;
      if (REPL) {
        sh_loc[l] = 0;
        sh0_loc[l] = 0;
        chg_loc[l] = 0;
        comp_loc[l] = l < Li ? (unsigned short)lcomp[l] : 0;
      }
      if (AGG) {
        dcap_loc[l] = 0;
        dn_loc[l] = 0;
      }
    }
    for (int s = tid; s < Sc; s += NT) {
      S.bn[s] = -3;
      S.tc[s] = kInf;
    }
    if (tid < M_NCTL) ctl[tid] = 0;
    if (crank == 0 && tid == 0) comb.ev_rounds = 0;
    __syncthreads();
    }

    auto fill_slot = [&](int slot, int out, const FlowRec &r, double ta) {
      S.flow[slot] = out;  // where the flow's results go
      S.rem[slot] = r.bytes;
      S.bn[slot] = -2;
      S.comp[slot] = (unsigned short)r.comp;
#pragma unroll
      for (int h = 0; h < kMaxHops; ++h)
        S.path[slot * kMaxHops + h] = r.path[h] < 0 ? kNoLink : (unsigned short)r.path[h];
      S.succ_cnt[slot] = r.succ_cnt;
      S.succ0[slot] = r.succ_in[0];
      S.succ1[slot] = r.succ_in[1];
      S.tc[slot] = ta;
    };

    // S4: outstanding predecessors.  Flows without predecessors are PENDING from t = 0 with t_act = start + Lat; they
    // wait in the unit's list sorted by t_act (built by phs_finalize) and take a slot only when they activate.
    if (!resuming)
      for (int64_t f = ctid; f < F; f += CT) pred_cnt[f] = pc0[f];
    const double *__restrict__ init_t = T.init_t + D.init_base;
    const int32_t *__restrict__ init_f = T.init_f + D.init_base;
    const int n_init = D.n_init;
    int ip = 0;  // entries [0, ip) of the list have been activated (the same in every thread of the cluster)
    double t_init = n_init > 0 ? __ldg(&init_t[0]) : kInf;
    if (resuming) {  // this CTA's shared memory, control words and cold slot fields as they were when the unit stopped
      const uint4 *src = (const uint4 *)cpark;
      uint4 *dst = (uint4 *)smem_raw;
      for (size_t i = tid; i < smem_used / 16; i += NT) dst[i] = src[i];
      const int *pctl = (const int *)(cpark + smem_used);
      if (tid < M_NCTL) ctl[tid] = pctl[tid];
      if (crank == 0 && tid == 0) comb = *(const Comb *)(cpark + smem_used + 64);
      if (!SC.cold_smem) {
        const uint4 *cs = (const uint4 *)(cpark + smem_used + 64 + sizeof(Comb));
        uint4 *cd = (uint4 *)S.rem;
        for (size_t i = tid; i < ((size_t)Sc * kSlotColdBytes + 15) / 16; i += NT) cd[i] = cs[i];
      }
    }
    __threadfence();  // pred_cnt[] is decremented by other CTAs of the cluster
    cluster.sync();

    double now = 0.0, t_next = 0.0;
    int ev = -1, solve = 0, g = 0;
    long long sum_active = 0, sum_rounds = 0;
    int max_active = 0, max_pending = 0, max_slots = 0;
    int status = PHS_OK;
    int first_bneck = -1;
#ifdef PHS_PHASE_CLOCKS
    long long pc_[8] = {0, 0, 0, 0, 0, 0, 0, 0}, pt_ = clock64();
#define PHS_TICK(i) { const long long t_ = clock64(); pc_[i] += t_ - pt_; pt_ = t_; }
#else
#define PHS_TICK(i)
#endif
    int nDone = 0, prev_nact = 0;
    double acc_min = kInf;  // (thread 0 of a CTA) minimum of the times folded in this event's rounds
    if (resuming) {
      const ClusterParkRegs *pr = (const ClusterParkRegs *)upark;
      now = pr->now; t_next = pr->t_next; t_init = pr->t_init;
      sum_active = pr->sum_active; sum_rounds = pr->sum_rounds;
      ev = pr->ev; solve = pr->solve; g = pr->g; ip = pr->ip; nDone = pr->n_done; prev_nact = pr->prev_nact;
      max_active = pr->max_active; max_pending = pr->max_pending; max_slots = pr->max_slots;
      first_bneck = pr->first_bneck;
    }

    // this CTA's slot high-water mark and free-queue tail as the next phase X must see them: read where a barrier
    // protects the read (here and after the X barrier of every event), never at the top of phase X, where warps
    // that are already inside the phase bump both words
    int hi_carry = min(ctl[M_HI], Sc), qtail_carry = ctl[M_QTAIL];

    for (;;) {
      if (t_next > T.t_stop) {  // phs_run_until: the next event lies beyond the requested time
        status = kPaused;
        break;
      }
      // ======== phase X (a8 + a4): retire what completes at t_next, release successors, activate what is due
      ++solve;
      const int hi0 = hi_carry;
      const int qtail = qtail_carry;
      auto touch_link = [&](int l, int delta) {  // the link's flow count changes: its share0 is stale for this solve
        LinkA *a = LA(l);
        atomicAdd(&a->n0, delta);
        a->chg = solve;
        if (REPL && !INC)
          for (int r = 0; r < CS; ++r) cluster.map_shared_rank(chg_loc, (unsigned)r)[l] = solve;
      };
      auto mark_comp = [&](int c) {  // the component must be re-solved: tell every CTA
        for (int r = 0; r < CS; ++r) cluster.map_shared_rank(csolve, (unsigned)r)[c] = solve;
      };
      auto limit_comp = [&](int c, long long rq) {  // INC: flows of component c with a rate >= rq must be re-solved
        const unsigned key = (unsigned)(rq >> kRminShift);
        for (int r = 0; r < CS; ++r) atomicMin(cluster.map_shared_rank(crmin, (unsigned)r) + c, key);
      };
      auto activate = [&](int slot) {
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {
          const int l = S.path[slot * kMaxHops + h];
          if (l == kNoLink) break;
          touch_link(l, 1);
        }
        mark_comp(S.comp[slot]);
        if (INC) ctl[M_ADDED] = 1;  // a flow was added: its links bound what stands (pass A after the X barrier)
        S.rq[slot] = -1;
        S.bn[slot] = -1;
        S.tc[slot] = kInf;
        atomicAdd(&ctl[M_NACT], 1);
        atomicSub(&ctl[M_NPEND], 1);
        if (LOG) atomicAdd(&ctl[M_EVA], 1);
        const int nsucc = S.succ_cnt[slot];  // the successors' records will be needed: pull them towards L2
        if (nsucc > 0 && nsucc <= 2) {
          asm volatile("prefetch.global.L2 [%0];" ::"l"(rec + S.succ0[slot]));
          if (nsucc > 1) asm volatile("prefetch.global.L2 [%0];" ::"l"(rec + S.succ1[slot]));
        }
      };
      auto make_pending = [&](int out, const FlowRec &r) {  // S4.5: t_act = max(start, now) + Lat
        const double ta = __dadd_rn(r.start > t_next ? r.start : t_next, r.lat);
        const int h = atomicAdd(&ctl[M_QHEAD], 1);
        const int slot = h < qtail ? S.freeq[h % Sc] : atomicAdd(&ctl[M_HI], 1);
        if (slot >= Sc) {
          ctl[M_OVER] = 1;
          return;
        }
        atomicAdd(&ctl[M_NPEND], 1);
        const bool due = ta <= t_next;
        fill_slot(slot, out, r, due ? kInf : ta);
        if (due) activate(slot);
      };
      auto release2 = [&](int g0, int g1) {  // both counters, then both records: the round trips overlap
        const bool z0 = g0 >= 0 && atomicSub(&pred_cnt[g0], 1) == 1;
        const bool z1 = g1 >= 0 && atomicSub(&pred_cnt[g1], 1) == 1;
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
        if (z0) make_pending(o0, r0);
        if (z1) make_pending(o1, r1);
      };
      for (int s = tid; s < hi0; s += NT) {
        if (!(S.tc[s] <= t_next)) continue;
        if (S.bn[s] == -2) {
          activate(s);
          continue;
        }
        const int f = S.flow[s];
        t_done[f] = t_next;
        bneck_out[f] = linkid[S.bn[s]];
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {
          const int l = S.path[s * kMaxHops + h];
          if (l == kNoLink) break;
          touch_link(l, -1);
          if (INC) add64_2x32(&LB(l)->caprem, S.rq[s]);  // the flow's rate goes back to its links
        }
        mark_comp(S.comp[s]);
        if (INC) limit_comp(S.comp[s], S.rq[s]);
        S.bn[s] = -3;
        S.tc[s] = kInf;
        S.freeq[atomicAdd(&ctl[M_QTAIL], 1) % Sc] = s;
        atomicSub(&ctl[M_NACT], 1);
        atomicAdd(&ctl[M_NDONE], 1);
        if (LOG) atomicAdd(&ctl[M_EVC], 1);
        const int nsucc = S.succ_cnt[s];
        if (nsucc <= 2) {
          if (nsucc > 0) release2(S.succ0[s], nsucc > 1 ? S.succ1[s] : -1);
        } else {
          const int e0 = S.succ0[s];
          for (int e = 0; e < nsucc; ++e) release2(succ[e0 + e], -1);
        }
      }
      // flows without predecessors whose time has come: entry k of the sorted list is taken by CTA k mod CS
      while (t_init <= t_next) {  // uniform over the cluster
        const int k = ip + tid;
        const bool due = k < n_init && __ldg(&init_t[k]) <= t_next;
        if (due && (k & cmask) == crank) {
          const int f = __ldg(&init_f[k]);
          const FlowRec r = rec[f];
          const int h = atomicAdd(&ctl[M_QHEAD], 1);
          const int slot = h < qtail ? S.freeq[h % Sc] : atomicAdd(&ctl[M_HI], 1);
          if (slot >= Sc) {
            ctl[M_OVER] = 1;
          } else {
            atomicAdd(&ctl[M_NPEND], 1);  // activate() moves it from PENDING to ACTIVE
            fill_slot(slot, (int)fmap[f], r, kInf);
            activate(slot);
          }
        }
        const int cnt = __syncthreads_count(due);
        ip += cnt;
        t_init = ip < n_init ? __ldg(&init_t[ip]) : kInf;
        if (cnt < NT) break;
      }
      PHS_TICK(0)
      __syncthreads();
      if (warp == 0) {  // publish this CTA's counts: lane r writes them into CTA r's own table (no read trip later)
        CombX x;
        x.n_act = ctl[M_NACT]; x.n_pend = ctl[M_NPEND]; x.n_done = ctl[M_NDONE]; x.over = ctl[M_OVER];
        x.hi = ctl[M_HI]; x.ev_ncomp = ctl[M_EVC]; x.ev_nact = ctl[M_EVA]; x.pad = ctl[M_ADDED];
        if (lane < CS) cluster.map_shared_rank(&comb, (unsigned)lane)->x[crank] = x;
        __syncwarp();
        if (lane == 0) {
          ctl[M_EVC] = 0;
          ctl[M_EVA] = 0;
          ctl[M_ADDED] = 0;
          if (ctl[M_QHEAD] > qtail) ctl[M_QHEAD] = qtail;
          ctl[M_NWL0] = 0;
          ctl[M_NWL1] = 0;
        }
      }
      PHS_TICK(1)
      cluster.sync();  // ---------------------------------------------------------------- cluster barrier X
      PHS_TICK(2)
      now = t_next;
      if (warp == 0) {  // one warp per CTA sums the per-CTA counts and hands them to the CTA
        CombX x;
        x.n_act = x.n_pend = x.n_done = x.over = x.hi = x.ev_ncomp = x.ev_nact = x.pad = 0;
        if (lane < CS) x = comb.x[lane];
        const int added = __reduce_or_sync(0xffffffffu, x.pad);
        const int a = __reduce_add_sync(0xffffffffu, x.n_act), b = __reduce_add_sync(0xffffffffu, x.n_pend);
        const int c = __reduce_add_sync(0xffffffffu, x.n_done), d = __reduce_add_sync(0xffffffffu, x.over);
        const int e = __reduce_max_sync(0xffffffffu, x.hi);
        const int nc = __reduce_add_sync(0xffffffffu, x.ev_ncomp), na = __reduce_add_sync(0xffffffffu, x.ev_nact);
        if (lane == 0) {
          bc[0] = a; bc[1] = b; bc[2] = c; bc[3] = d; bc[4] = e; bc[5] = nc; bc[6] = na; bc[8] = added;
        }
      }
      __syncthreads();
      const int nA = bc[0], nPend = bc[1] + (n_init - ip), over = bc[3];
      nDone = bc[2];
      max_slots = max(max_slots, bc[4]);
      if (LOG && ctid == 0) {
        if (log && ev >= 0) {  // O4: the event that just finished
          phs_event e;
          e.t = now;
          e.n_completed = bc[5];
          e.n_activated = prev_nact;
          e.n_rounds = comb.ev_rounds;
          e.first_bneck = first_bneck;
          log[ev] = e;
        }
        comb.ev_rounds = 0;
        prev_nact = bc[6];
      }
      ++ev;
      if (over) {
        status = kOverflow;
        break;
      }
      if (nA == 0 && nPend == 0) break;
      const int hi = hi_carry = min(ctl[M_HI], Sc);
      qtail_carry = ctl[M_QTAIL];
      max_active = max(max_active, nA);
      max_pending = max(max_pending, nPend);

      if (INC && bc[8]) {
        // ======== A: flows were ADDED in this event.  A link that carries an added flow has a share of at least
        // floor(cap / n) -- n its flow count now -- all through the new solve, so the old solve's iterations below the
        // smallest such share are picked again in the same order: every flow slower than that stands.
        for (int s = tid; s < hi; s += NT) {
          if (S.bn[s] != -1 || S.rq[s] >= 0) continue;  // ACTIVE and never solved = added
          long long m = LLONG_MAX;
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {
            const int l = S.path[s * kMaxHops + h];
            if (l == kNoLink) break;
            const LinkA *ap = LA(l);
            const long long sh = fair_share(ap->cap, ap->n0);
            m = sh < m ? sh : m;
          }
          limit_comp(S.comp[s], m);
        }
        cluster.sync();  // ---------------------------------------------------------------- cluster barrier A
      }
      // ======== P: working capacities of the own links that will be re-solved (first debited after barrier 1)
      if (!INC)
      for (int li = tid; li < Lc; li += NT) {
        if (LOG || csolve[lb[li].comp] == solve) {
          lb[li].caprem = la[li].cap;
          lb[li].nw = la[li].n0;
        }
      }
      if (REPL && !INC) {
        for (int l = tid; l < L; l += NT)
          if (LOG || csolve[comp_loc[l]] == solve) sh_loc[l] = sh0_loc[l];
        __syncthreads();
      }

      // ======== rates (a5-a7): parallel progressive filling over the components this event touched
      unsigned short *wl = S.wl0, *wl_next = S.wl1;
      int nwl_idx = M_NWL0;
      double mymin = kInf;  // completion / activation times of this thread's flows, folded as they become final
      // a5 + a6: the fair share of every link of the flow's path, refreshed by the flow itself where it is stale
      // (every flow on such a link computes and stores the same value), arg-min (share, id), beat the other links
      auto vote = [&](int s, bool first) {
        int p[kMaxHops];
        long long sh[kMaxHops];
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {  // all loads first: one DSMEM round trip for the whole path
          const int l = p[h] = S.path[s * kMaxHops + h];
          sh[h] = LLONG_MAX;
          if (l == kNoLink) continue;
          if (REPL) {
            if (first && chg_loc[l] == solve) {  // flow count changed in this event: fetch it from the owner
              LinkA *ap = LA(l);
              const long long cap = ap->cap;
              const int n0 = ap->n0;
              sh[h] = fair_share(cap, n0);
              sh0_loc[l] = sh[h];
              sh_loc[l] = sh[h];
            } else {
              sh[h] = sh_loc[l];
            }
            continue;
          }
          LinkA *ap = LA(l);
          const longlong2 a = *(const longlong2 *)ap;         // share0, cap
          const int4 ai = *((const int4 *)ap + 1);            // n0, chg, beat, solve
          if (first) {
            if (ai.y == solve) {  // flow count changed in this event
              sh[h] = fair_share(a.y, ai.x);
              ap->share0 = sh[h];
            } else {
              sh[h] = a.x;
            }
          } else {
            LinkB *bp = LB(l);
            const longlong2 b = *(const longlong2 *)bp;       // caprem, sharew
            const int4 bi = *((const int4 *)bp + 1);          // nw, deb, wsolve, comp
            if (bi.y == g - 1) {  // debited in the previous round
              sh[h] = fair_share(b.x, bi.x);
              bp->sharew = sh[h];
              bp->wsolve = solve;
            } else {
              sh[h] = bi.z == solve ? b.y : a.x;
            }
          }
        }
        long long best = LLONG_MAX;
        int arg = -1;
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h)
          if (p[h] != kNoLink && (sh[h] < best || (sh[h] == best && p[h] < arg))) {
            best = sh[h];
            arg = p[h];
          }
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h)
          if (p[h] != kNoLink && p[h] != arg && beatf[p[h]] != g) {  // one stamp per link, CTA and round
            beatf[p[h]] = g;
            LA(p[h])->beat = g;
          }
        S.arg[s] = (unsigned short)arg;
        return make_longlong2(best, (long long)arg);
      };
      auto freeze = [&](int s, int arg, long long rq) {  // a7 + R-LZ settle
        S.bn[s] = arg;
        const long long old = S.rq[s];
        if (rq != old) {
          double rem = S.rem[s];
          if (old >= 0) {
            rem = __dsub_rn(rem, __dmul_rn(rate_of(old), __dsub_rn(now, S.tl[s])));
            rem = rem > 0.0 ? rem : 0.0;
            S.rem[s] = rem;
          }
          S.tl[s] = now;
          S.rq[s] = rq;
          if (T.hist) append_history(T.hist, T.hist_n, T.hist_cap, now, rq, (uint32_t)S.flow[s], (uint32_t)ev);
          S.tc[s] = __dadd_rn(now, __ddiv_rn(rem, rate_of(rq)));
        }
        mymin = dmin(mymin, S.tc[s]);
        if (LOG && atomicExch(cluster.map_shared_rank(won + (arg >> csh), (unsigned)(arg & cmask)), g) != g)
          atomicAdd(&comb0->ev_rounds, 1);
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {  // debit the path
          const int l = S.path[s * kMaxHops + h];
          if (l == kNoLink) break;
          if (AGG) {
            if (atomicAdd(&dn_loc[l], 1) == 0) touched[atomicAdd(&ctl[M_NTOUCH], 1)] = l;
            add64_2x32(&dcap_loc[l], rq);
          } else {
            LinkB *bp = LB(l);
            add64_2x32(&bp->caprem, -rq);
            atomicSub(&bp->nw, 1);
            bp->deb = g;
          }
        }
      };

      int rounds = 0;
      ++g;
      {  // ---- V0: collect the flows to re-solve, vote; fold the times of everybody else
        long long bk = LLONG_MAX;
        int bl = INT_MAX;
        for (int s = tid; s < hi; s += NT) {
          const int bn0 = S.bn[s];
          if (bn0 == -3) continue;
          bool in = bn0 != -2 && (LOG || csolve[S.comp[s]] == solve);
          if (INC && in) {  // rates below the smallest removed rate stand (never solved: rq = -1, always in)
            const long long rq = S.rq[s];
            in = rq < 0 || (unsigned)(rq >> kRminShift) >= crmin[S.comp[s]];
          }
          if (!in) {
            mymin = dmin(mymin, S.tc[s]);
            continue;
          }
          S.bn[s] = -1;
          wl[atomicAdd(&ctl[nwl_idx], 1)] = (unsigned short)s;
          if (INC) {  // the flow's rate goes back to its links, which count it as unfrozen again (pre-summed per CTA)
            const long long rq = S.rq[s];
#pragma unroll
            for (int h = 0; h < kMaxHops; ++h) {
              const int l = S.path[s * kMaxHops + h];
              if (l == kNoLink) break;
              if (atomicAdd(&dn_loc[l], 1) == 0) touched[atomicAdd(&ctl[M_NTOUCH], 1)] = l;
              if (rq > 0) add64_2x32(&dcap_loc[l], rq);
            }
            continue;  // the vote follows once the owners have the links' new shares
          }
          const longlong2 v = vote(s, true);
          if (LOG && (v.x < bk || (v.x == bk && (int)v.y < bl))) {
            bk = v.x;
            bl = (int)v.y;
          }
        }
        if (LOG) {  // first_bneck: per-CTA partial, combined by thread 0 of the cluster later
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
            red_key[warp] = bk;
            red_id[warp] = bl;
          }
          __syncthreads();
          if (tid == 0) {
            for (int w = 1; w < NT / 32; ++w)
              if (red_key[w] < bk || (red_key[w] == bk && red_id[w] < bl)) {
                bk = red_key[w];
                bl = red_id[w];
              }
            comb0->f[crank].fb_key = bk;
            comb0->f[crank].fb_id = bl;
          }
        }
      }
      if (INC) {
        // ---- C: credits to the owners (stamp deb = g marks the links whose share must be computed)
        __syncthreads();
        {
          const int nt = ctl[M_NTOUCH];
          for (int i = tid; i < nt; i += NT) {
            const int l = touched[i];
            LinkB *bp = LB(l);
            if (dcap_loc[l] != 0) add64_2x32(&bp->caprem, dcap_loc[l]);
            atomicAdd(&bp->nw, dn_loc[l]);
            bp->deb = g;
            dcap_loc[l] = 0;
            dn_loc[l] = 0;
          }
        }
        for (int c = tid; c < L; c += NT)  // this CTA has read its limits: ready for the next event
          if (csolve[c] == solve) crmin[c] = 0xffffffffu;
        __syncthreads();
        if (tid == 0) ctl[M_NTOUCH] = 0;
        cluster.sync();  // ---------------------------------------------------------------- cluster barrier C
        // ---- R0: owners compute the share of their credited links and tell every CTA
        for (int li = tid; li < Lc; li += NT) {
          if (lb[li].deb != g) continue;
          const int nw = lb[li].nw;
          if (nw <= 0) continue;
          const long long shv = fair_share(lb[li].caprem, nw);
          const int l = li * CS + crank;
          for (int r = 0; r < CS; ++r) cluster.map_shared_rank(sh_loc, (unsigned)r)[l] = shv;
        }
        cluster.sync();  // ---------------------------------------------------------------- cluster barrier R0
        ++g;
        const int nv = ctl[nwl_idx];
        for (int i = tid; i < nv; i += NT) vote(wl[i], false);
      }
      for (;;) {
        PHS_TICK(3)
        cluster.sync();  // -------------------------------------------------------------- cluster barrier 1
        PHS_TICK(4)
        ++rounds;
        // ---- F: flows whose arg-min link is unbeaten freeze (a7), settle (R-LZ) and debit; the rest stay listed
        const int nwl = ctl[nwl_idx];
        const int nxt_idx = nwl_idx == M_NWL0 ? M_NWL1 : M_NWL0;
        bool left = false;
        for (int i = tid; i < nwl; i += NT) {
          const int s = wl[i];
          const int arg = S.arg[s];
          LinkA *ap = LA(arg);
          const long long share0 = REPL ? sh_loc[arg] : ap->share0;
          const int beat = ap->beat;
          long long rq = share0;
          if (!REPL && rounds > 1) {
            LinkB *bp = LB(arg);
            const long long sw = bp->sharew;
            if (bp->wsolve == solve) rq = sw;
          }
          if (beat != g) {
            freeze(s, arg, rq);
          } else {
            wl_next[atomicAdd(&ctl[nxt_idx], 1)] = (unsigned short)s;
            left = true;
          }
        }
        const double wm = warp_min(mymin);
        if (lane == 0) red[warp] = wm;
        left = __syncthreads_or(left);
        // ---- combine: this CTA's debits, its minimum time and its "flows left" flag
        if (AGG) {
          const int nt = ctl[M_NTOUCH];
          for (int i = tid; i < nt; i += NT) {
            const int l = touched[i];
            LinkB *bp = LB(l);
            add64_2x32(&bp->caprem, -dcap_loc[l]);
            atomicSub(&bp->nw, dn_loc[l]);
            bp->deb = g;
            dcap_loc[l] = 0;
            dn_loc[l] = 0;
          }
        }
        if (warp == 0) {
          const double m = warp_min(lane < NT / 32 ? red[lane] : kInf);
          if (lane < CS) {  // lane r tells CTA r
            CombF *cf = &cluster.map_shared_rank(&comb, (unsigned)lane)->f[crank];
            cf->tmin = m;
            cf->left = left ? 1 : 0;
          }
        }
        PHS_TICK(5)
        cluster.sync();  // -------------------------------------------------------------- cluster barrier 2
        PHS_TICK(6)
        if (warp == 0) {
          double m = kInf;
          int lf = 0;
          if (lane < CS) {
            m = comb.f[lane].tmin;
            lf = comb.f[lane].left;
          }
          m = warp_min(m);
          lf = __reduce_or_sync(0xffffffffu, lf);
          if (lane == 0) {
            bc_t = acc_min = dmin(acc_min, m);
            bc[7] = lf;
            ctl[nwl_idx] = 0;
            ctl[M_NTOUCH] = 0;
          }
        }
        mymin = kInf;  // folded
        __syncthreads();
        if (!bc[7]) break;
        if (REPL) {  // ---- R: owners recompute the share of their links debited in this round and tell every CTA
          for (int li = tid; li < Lc; li += NT) {
            if (lb[li].deb != g) continue;
            const int nw = lb[li].nw;
            if (nw <= 0) continue;
            const long long shv = fair_share(lb[li].caprem, nw);
            const int l = li * CS + crank;
            for (int r = 0; r < CS; ++r) cluster.map_shared_rank(sh_loc, (unsigned)r)[l] = shv;
          }
          cluster.sync();  // ------------------------------------------------------------ cluster barrier 3
        }
        // ---- V: the flows still listed vote on the new shares
        ++g;
        {
          unsigned short *t = wl;
          wl = wl_next;
          wl_next = t;
          nwl_idx = nxt_idx;
        }
        const int nv = ctl[nwl_idx];
        for (int i = tid; i < nv; i += NT) vote(wl[i], false);
      }
      // ======== next time (a8)
      t_next = dmin(bc_t, t_init);
      acc_min = kInf;
      if (LOG && ctid == 0) {
        first_bneck = -1;
        if (nA > 0) {
          long long bk = LLONG_MAX;
          for (int c = 0; c < CS; ++c) {
            const long long k = comb.f[c].fb_key;
            const int id = comb.f[c].fb_id;
            if (k < bk || (k == bk && id < first_bneck)) {
              bk = k;
              first_bneck = id;
            }
          }
        }
      }
      sum_active += nA;
      sum_rounds += rounds;
    }
    if (upark) {  // park the unit if it stopped at t_stop; a finished unit has nothing to resume
      if (status == kPaused) {
        __syncthreads();
        uint4 *dst = (uint4 *)cpark;
        const uint4 *src = (const uint4 *)smem_raw;
        for (size_t i = tid; i < smem_used / 16; i += NT) dst[i] = src[i];
        int *pctl = (int *)(cpark + smem_used);
        if (tid < M_NCTL) pctl[tid] = ctl[tid];
        if (crank == 0 && tid == 0) *(Comb *)(cpark + smem_used + 64) = comb;
        if (!SC.cold_smem) {
          uint4 *cd = (uint4 *)(cpark + smem_used + 64 + sizeof(Comb));
          const uint4 *cs = (const uint4 *)S.rem;
          for (size_t i = tid; i < ((size_t)Sc * kSlotColdBytes + 15) / 16; i += NT) cd[i] = cs[i];
        }
      }
      if (ctid == 0) {
        ClusterParkRegs r;
        r.now = now; r.t_next = t_next; r.t_init = t_init; r.sum_active = sum_active; r.sum_rounds = sum_rounds;
        r.ev = ev; r.solve = solve; r.g = g; r.ip = ip; r.n_done = nDone; r.prev_nact = prev_nact;
        r.max_active = max_active; r.max_pending = max_pending; r.max_slots = max_slots; r.first_bneck = first_bneck;
        r.valid = status == kPaused ? 1 : 0; r.pad_ = 0;
        *(ClusterParkRegs *)upark = r;
      }
    }
#ifdef PHS_PHASE_CLOCKS
    if (tid == 0 && (crank == 0 || crank == CS - 1))
      printf("inst %d cta %d/%d events %d cycles: X %lld pub %lld barX %lld P+V %lld bar1 %lld F %lld bar2 %lld\n", inst, crank,
             CS, ev, pc_[0], pc_[1], pc_[2], pc_[3], pc_[4], pc_[5], pc_[6]);
#endif
    if (ctid == 0) {
      InstResult r;
      r.status = status != PHS_OK ? status : (nDone < F ? PHS_ECYCLE : PHS_OK);
      r.path = 1;
      r.n_events = ev;
      r.sum_active = sum_active;
      r.sum_par_rounds = sum_rounds;
      r.max_active = max_active;
      r.max_pending = max_pending;
      r.max_slots = max_slots;
      r.n_windows = ev;  // one event per iteration on this path
      T.res[inst] = r;
    }
    cluster.sync();
  }
}

// ------------------------------------------------------------------------------------------------ launch
namespace {
void set_cluster_attr(cudaLaunchConfig_t &cfg, cudaLaunchAttribute *attr, int cluster_size, int n_clusters,
                      size_t smem, cudaStream_t stream) {
  cfg.gridDim = dim3((unsigned)(cluster_size * n_clusters));
  cfg.blockDim = dim3(kClusterThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)cluster_size;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
}

template <bool LOG, bool AGG>
cudaError_t prepare(size_t smem) {
  cudaError_t e = cudaFuncSetAttribute(phs_cluster_kernel<LOG, AGG>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(phs_cluster_kernel<LOG, AGG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}

template <bool LOG, bool AGG>
cudaError_t launch_cluster_t(const DevTables &t, const int32_t *list, int n, int *ticket, const ClusterScratch &s,
                             int cluster_size, int n_clusters, cudaStream_t stream) {
  const size_t smem = cluster_smem_bytes(t.n_links, cluster_size, s.Sc, AGG, s.cold_smem != 0, LOG, s.replicate != 0);
  cudaError_t e = prepare<LOG, AGG>(smem);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute attr[1];
  set_cluster_attr(cfg, attr, cluster_size, n_clusters, smem, stream);
  return cudaLaunchKernelEx(&cfg, phs_cluster_kernel<LOG, AGG>, t, list, n, ticket, s);
}
}  // namespace

cudaError_t launch_cluster_path(const DevTables &t, const int32_t *list, int n, int *ticket, const ClusterScratch &s,
                                int cluster_size, int n_clusters, bool log, cudaStream_t stream) {
  if (s.aggregate)
    return log ? launch_cluster_t<true, true>(t, list, n, ticket, s, cluster_size, n_clusters, stream)
               : launch_cluster_t<false, true>(t, list, n, ticket, s, cluster_size, n_clusters, stream);
  return log ? launch_cluster_t<true, false>(t, list, n, ticket, s, cluster_size, n_clusters, stream)
             : launch_cluster_t<false, false>(t, list, n, ticket, s, cluster_size, n_clusters, stream);
}

cudaError_t cluster_max_clusters(int cluster_size, size_t smem, int *max_clusters) {
  cudaError_t e = prepare<true, true>(smem);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute attr[1];
  set_cluster_attr(cfg, attr, cluster_size, 1, smem, nullptr);
  int n = 0;
  e = cudaOccupancyMaxActiveClusters(&n, phs_cluster_kernel<true, true>, &cfg);
  if (e != cudaSuccess) {
    (void)cudaGetLastError();
    n = 0;
  }
  *max_clusters = n;
  return cudaSuccess;
}

}  // namespace phs
