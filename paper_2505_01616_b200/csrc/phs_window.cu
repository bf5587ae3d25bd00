// phs_window.cu -- window path of the hot path: the lookahead-window schedule (conservative parallel discrete-event
// simulation over static link components), for units whose events are dense in simulated time.
// a4-a9; same rate arithmetic and phases as the CTA path (phs_kernels.cu), different event schedule.
//
// Why it is exact ("Lookahead windows").  Under reading R-LZ a flow's state changes only when its
// own rate changes, and rates are a function of the ACTIVE set of the flow's static link component; components
// influence each other only through DAG releases, and a flow released by a completion at time t becomes ACTIVE at
// max(start, t) + Lat >= t + lmin, lmin = the smallest path latency among the unit's dependent flows.  Let T0 be the
// earliest pending event of the unit.  No release produced at or after T0 can take effect before T0 + lmin, so inside
// the window [T0, T0 + lmin) every component evolves on its own: one loop iteration processes the NEXT event of
// EVERY component that has one inside the window, each at its own time (c_next / c_now per component), and the
// successors of the window's completions are created once, at the end of the window (phase R), with
// t_act = max(start, latest predecessor) + Lat.  Every flow sees exactly the solves, at exactly the times, that the
// one-event-per-iteration schedule gives it, so completion times, bottlenecks and order are bit-identical; the
// dependent chain shrinks from the number of distinct event times to the number of window iterations (BASELINE.json
// configs[2]: 1.83 M events -> 20.6 K windows / 54.8 K iterations).
//
// Gang of K CTAs (one thread-block cluster, K = 1, 2, 4, 8, 16).  Components never share state inside a window, so
// they are PARTITIONED over the CTAs of the cluster: CTA k owns a set of components with their links and the slots
// of their flows, all in its own shared memory, and runs its iterations without talking to anybody.  Only at the end
// of a window do the CTAs meet: cluster barrier, every CTA reads the release lists of all CTAs through distributed
// shared memory and creates the slots of the flows it owns, cluster barrier, next T0 = min over the CTAs.
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include <climits>

#include "phs_device.h"
#include "phs_devutil.cuh"

namespace cg = cooperative_groups;

namespace phs {

namespace {

constexpr int NT = kWindowThreads;
constexpr int NW = NT / 32;
constexpr unsigned kNoLink = 0xffffu;
constexpr unsigned kLocMask = 0xffffffu;  // lloc / cown / fown: owner << 24 | index local to the owner

struct WinSmem {
  // per own link [L]
  long long *l_cap, *l_share0, *l_caprem, *l_sharew;
  int *l_n0, *l_chg, *l_beat, *l_nw, *l_deb, *l_gid;
  // per own component [NC]
  int *c_solve;    // id of the iteration whose solve must redo the component
  double *c_next;  // time of the component's next event = min over its slots of s_tc
  double *c_now;   // time of the event the component processes in the current iteration
  // per slot [S]: one slot per PENDING or ACTIVE flow of an own component
  double *s_tc, *s_rem, *s_tl;
  long long *s_rq;
  int4 *s_meta;    // .x output position (-1 = free); .y -2 PENDING, -1 ACTIVE unfrozen, >= 0 bottleneck (own link index);
                   // .z own component index; .w arg-min link of the current round
  uint4 *s_path;   // own link indices, 8 x uint16
  int *s_succ_cnt, *s_succ0, *s_succ1;
  int *free_q;
  // release list [RLC]: successor releases of the current window (unit-local flow ids; the completion time goes
  // into the flow's word of the global array t_rel by atomic max)
  int *rl_flow;
  int *chg_list;   // [CLC] links whose flow count changed in the current iteration (duplicates allowed)
  double *red;     // [32]
  double *red2;    // [32]
  int *ctl;        // [32]
};
enum { C_HI = 0, C_QHEAD, C_QTAIL, C_NACTIVE, C_NPEND, C_OVERFLOW, C_DONE, C_NRL, C_NCHG, C_NCTL };

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
__host__ __device__ inline int rl_capacity(int slots) { return 2 * slots + 64; }
// changed-link list: 6 links per flow that fires; an iteration that overflows it falls back to a scan of all links
__host__ __device__ inline int chg_capacity(int slots) { return slots < 256 ? 256 : slots; }

__host__ __device__ inline size_t carve(WinSmem *s, unsigned char *base, int L, int NC, int S) {
  size_t o = 0, a;
#define PHS_TAKE(field, type, count)                    \
  a = o;                                                \
  o = align_up(o + sizeof(type) * (size_t)(count), 16); \
  if (s) s->field = (type *)(base + a);
  PHS_TAKE(l_cap, long long, L)
  PHS_TAKE(l_share0, long long, L)
  PHS_TAKE(l_caprem, long long, L)
  PHS_TAKE(l_sharew, long long, L)
  PHS_TAKE(c_next, double, NC)
  PHS_TAKE(c_now, double, NC)
  PHS_TAKE(s_tc, double, S)
  PHS_TAKE(s_rem, double, S)
  PHS_TAKE(s_tl, double, S)
  PHS_TAKE(s_rq, long long, S)
  PHS_TAKE(red, double, 32)
  PHS_TAKE(red2, double, 32)
  PHS_TAKE(l_n0, int, L)
  PHS_TAKE(l_chg, int, L)
  PHS_TAKE(l_beat, int, L)
  PHS_TAKE(l_nw, int, L)
  PHS_TAKE(l_deb, int, L)
  PHS_TAKE(l_gid, int, L)
  PHS_TAKE(c_solve, int, NC)
  PHS_TAKE(s_meta, int4, S)
  PHS_TAKE(s_path, uint4, S)
  PHS_TAKE(s_succ_cnt, int, S)
  PHS_TAKE(s_succ0, int, S)
  PHS_TAKE(s_succ1, int, S)
  PHS_TAKE(free_q, int, S)
  PHS_TAKE(rl_flow, int, rl_capacity(S))
  PHS_TAKE(chg_list, int, chg_capacity(S))
  PHS_TAKE(ctl, int, 32)
#undef PHS_TAKE
  return o;
}

__device__ __forceinline__ int path_at(const uint4 &p, int h) {
  const unsigned w = h < 2 ? p.x : h < 4 ? p.y : h < 6 ? p.z : p.w;
  return (int)((h & 1) ? (w >> 16) : (w & 0xffffu));
}

// 64-bit add on a shared-memory word with two native 32-bit atomics (exact once all adds of a phase completed)
__device__ __forceinline__ void smem_add64(long long *p, long long v) {
  unsigned *w = (unsigned *)p;
  const unsigned lo = (unsigned)(unsigned long long)v, hi = (unsigned)((unsigned long long)v >> 32);
  const unsigned old = atomicAdd(w, lo);
  const unsigned carry = (old + lo) < old ? 1u : 0u;
  if (hi + carry) atomicAdd(w + 1, hi + carry);
}

// min of a non-negative double into a shared-memory word (bit patterns order like unsigned integers); a plain read
// first, so that the common case -- nothing to lower -- issues no atomic
__device__ __forceinline__ void smem_min_f64(double *p, double v) {
  unsigned long long *q = (unsigned long long *)p;
  const unsigned long long nv = (unsigned long long)__double_as_longlong(v);
  unsigned long long old = *(volatile unsigned long long *)q;
  while (nv < old) {
    const unsigned long long prev = atomicCAS(q, old, nv);
    if (prev == old) break;
    old = prev;
  }
}

__device__ __forceinline__ double warp_min_nonneg(double v) {
  const unsigned long long b = (unsigned long long)__double_as_longlong(v);
  const unsigned hi = (unsigned)(b >> 32), lo = (unsigned)b;
  const unsigned mhi = __reduce_min_sync(0xffffffffu, hi);
  const unsigned mlo = __reduce_min_sync(0xffffffffu, hi == mhi ? lo : 0xffffffffu);
  return __longlong_as_double((long long)(((unsigned long long)mhi << 32) | mlo));
}

// what a CTA of the gang tells the others at the two barriers of a window end
struct Mailbox {
  double t_next;       // earliest event of the CTA's components (after phase R)
  int rl_base, rl_end; // release-list entries [rl_base, rl_end) of the window that just ended
  int live;            // ACTIVE + PENDING flows
  int over;            // ran out of slots or list entries
  int done;            // flows completed so far
  int iters;           // loop iterations so far
  long long sum_active, sum_rounds;
  int max_active, max_pending, max_slots, unit;
};

}  // namespace

size_t window_smem_bytes(int n_links, int n_comps, int slots) { return carve(nullptr, nullptr, n_links, n_comps, slots); }

// ================================================================================================ window kernel
__global__ void __launch_bounds__(kWindowThreads, 1)
    phs_window_kernel(DevTables T, const int32_t *__restrict__ list, int n_list, int *ticket, WindowLaunch W) {
  cg::cluster_group cluster = cg::this_cluster();
  const int K = (int)cluster.num_blocks();
  const int me = (int)cluster.block_rank();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ Mailbox mb;
  __shared__ int rl_lo[16], rl_n[16];  // phase R: first entry and length of every CTA's release list
  WinSmem S;
  const int SC = W.slots;
  carve(&S, smem_raw, W.n_links, W.n_comps, SC);
  const int RLC = rl_capacity(SC), CLC = chg_capacity(SC);
  Mailbox *mb0 = cluster.map_shared_rank(&mb, 0);

  for (;;) {
    // ---- a9: clusters pull units from the list
    if (me == 0 && tid == 0) mb.unit = atomicAdd(ticket, 1);
    cluster.sync();
    const int qi = mb0->unit;
    cluster.sync();
    if (qi >= n_list) break;
    const int inst = list[qi];
    const InstDesc D = T.inst[inst];
    const FlowRec *__restrict__ rec = T.rec + D.flow_base;
    const int32_t *__restrict__ succ = T.succ + D.succ_base;
    const int32_t *__restrict__ pc0 = T.pred_cnt0 + D.flow_base;
    int32_t *pred_cnt = T.pred_cnt + D.flow_base;
    const uint32_t *__restrict__ fmap = T.fmap + D.flow_base;
    const int64_t *__restrict__ capq = T.capq + D.link_base;
    const int32_t *__restrict__ linkid = T.linkid + D.link_base;
    const uint32_t *__restrict__ lloc = T.lloc + D.link_base;   // unit link -> owner << 24 | index in the owner
    const uint32_t *__restrict__ cown = T.cown + D.comp_base;   // unit component -> owner << 24 | index in the owner
    double *t_done = T.t_done;
    int32_t *bneck_out = T.bneck;
    const int F = D.n_flows;
    const double lmin = D.lmin;

    // ---- init: own links and components, every slot free, predecessor counters (split over the gang)
    for (int l = tid; l < D.n_links; l += NT) {
      const unsigned w = lloc[l];
      if ((int)(w >> 24) != me) continue;
      const int li = (int)(w & kLocMask);
      S.l_cap[li] = capq[l];
      S.l_gid[li] = linkid[l];
      S.l_n0[li] = 0;
      S.l_chg[li] = 0;
      S.l_beat[li] = 0;
      S.l_deb[li] = 0;
    }
    for (int c = tid; c < W.n_comps; c += NT) {
      S.c_solve[c] = 0;
      S.c_next[c] = kInf;
      S.c_now[c] = 0.0;
    }
    for (int s = tid; s < SC; s += NT) {
      S.s_meta[s].x = -1;
      S.s_tc[s] = kInf;
    }
    if (tid < C_NCTL) S.ctl[tid] = 0;
    unsigned long long *t_rel = T.t_rel + D.flow_base;  // per flow: latest completion among its predecessors so far
    uint32_t *fcw = T.fcw + D.flow_base;                 // per flow: owner << 24 | index of its component in the owner
    for (int f = me * NT + tid; f < F; f += K * NT) {
      pred_cnt[f] = pc0[f];
      t_rel[f] = 0ull;
      fcw[f] = cown[rec[f].comp];
    }
    __threadfence();  // all three are read / decremented by whichever CTA owns the flow
    __syncthreads();

    // one slot per PENDING or ACTIVE flow; link and component ids are translated to the owner's indices
    auto fill_slot = [&](int slot, int out, const FlowRec &r, double ta, int comp_local) {
      S.s_meta[slot].x = out;
      S.s_rem[slot] = r.bytes;
      S.s_meta[slot].y = -2;
      S.s_meta[slot].z = comp_local;
      {
        unsigned w[4] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0xffffffffu};
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {
          const unsigned l = r.path[h] < 0 ? kNoLink : (lloc[r.path[h]] & kLocMask);
          w[h >> 1] = (h & 1) ? ((w[h >> 1] & 0xffffu) | (l << 16)) : ((w[h >> 1] & 0xffff0000u) | l);
        }
        S.s_path[slot] = make_uint4(w[0], w[1], w[2], w[3]);
      }
      S.s_succ_cnt[slot] = r.succ_cnt;
      S.s_succ0[slot] = r.succ_in[0];
      S.s_succ1[slot] = r.succ_in[1];
      S.s_tc[slot] = ta;
    };

    // S4: flows without predecessors are PENDING from t = 0 with t_act = start + Lat.  They wait in the unit's list
    // sorted by t_act (built by phs_finalize) and take a slot, in the CTA that owns their component, at the start of
    // the window that contains t_act -- before any event of that window is processed.  `ip` entries are in slots;
    // every CTA of the gang advances it identically.
    const double *__restrict__ init_t = T.init_t + D.init_base;
    const int32_t *__restrict__ init_f = T.init_f + D.init_base;
    const int n_init = D.n_init;
    int ip = 0;
    double t_init = n_init > 0 ? __ldg(&init_t[0]) : kInf;

    double t_next = kInf;  // earliest event of this CTA's components
    int iters = 0, solve = 0, g = 0;
    long long sum_active = 0, sum_rounds = 0;
    int max_active = 0, max_pending = 0;
    int status = PHS_OK;
    // RULE: a control word is only read at a point that a barrier separates from every phase that writes it (right
    // after the X barrier of an iteration; after the barriers of the window start and end)
    int hi_c = 0, qtail_c = 0, nrl_c = 0, rl_base = 0, over_c = 0;
    const int NCw = W.n_comps;
    // earliest event of the own components = min over c_next (exact: every component folds its slots again whenever
    // one of them changes).  Few components: every thread reads them all; many: block reduction.
    auto next_event = [&]() {
      double m = kInf;
      if (NCw <= 64) {
        for (int c = 0; c < NCw; ++c) m = dmin(m, S.c_next[c]);
      } else {
        for (int c = tid; c < NCw; c += NT) m = dmin(m, S.c_next[c]);
        const double wm = warp_min_nonneg(m);
        if (lane == 0) S.red[warp] = wm;
        __syncthreads();
        m = S.red[0];
#pragma unroll
        for (int w = 1; w < NW; ++w) m = dmin(m, S.red[w]);
        __syncthreads();  // red[] is free again
      }
      return m;
    };
    if (tid == 0) {
      mb.t_next = kInf;
      mb.live = 0;
      mb.over = 0;
      mb.rl_base = mb.rl_end = 0;
    }
    cluster.sync();
    int n_windows = 0;
#ifdef PHS_PHASE_CLOCKS
    long long pc_[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, pt_ = clock64();
#define PHS_TICK(i) { const long long t_ = clock64(); pc_[i] += t_ - pt_; pt_ = t_; }
#else
#define PHS_TICK(i)
#endif

    for (;;) {  // ================================================================================ one window
      // ---- window start: T0 = min over the gang, everybody stops if somebody overflowed or nothing is left
      double T0 = t_init;
      int live = n_init - ip, over = 0;
      for (int k = 0; k < K; ++k) {
        const Mailbox *o = cluster.map_shared_rank(&mb, k);
        T0 = dmin(T0, o->t_next);
        live += o->live;
        over |= o->over;
      }
      if (over) {
        status = kOverflow;
        break;
      }
      if (live == 0) break;  // S4.3: nothing active, nothing pending -> stop
      const double wend = __dadd_rn(T0, lmin);  // window [T0, T0 + lmin)
      ++n_windows;
      // ---- initial flows whose t_act falls into the window take their slots now
      if (t_init < wend) {
        const int qt = qtail_c;
        for (;;) {
          const int k = ip + tid;
          const bool due = k < n_init && __ldg(&init_t[k]) < wend;
          if (due) {
            const int f = __ldg(&init_f[k]);
            const unsigned cw = __ldcg(&fcw[f]);
            if ((int)(cw >> 24) == me) {
              const FlowRec r = rec[f];
              const int h = atomicAdd(&S.ctl[C_QHEAD], 1);
              const int slot = h < qt ? S.free_q[h % SC] : atomicAdd(&S.ctl[C_HI], 1);
              if (slot < SC) {
                const double ta = __dadd_rn(r.start, r.lat);
                atomicAdd(&S.ctl[C_NPEND], 1);
                fill_slot(slot, (int)fmap[f], r, ta, (int)(cw & kLocMask));
                smem_min_f64(&S.c_next[cw & kLocMask], ta);
              } else {
                S.ctl[C_OVERFLOW] = 1;
              }
            }
          }
          const int cnt = __syncthreads_count(due);
          ip += cnt;
          t_init = ip < n_init ? __ldg(&init_t[ip]) : kInf;
          if (cnt < NT) break;
        }
        if (tid == 0 && S.ctl[C_QHEAD] > qt) S.ctl[C_QHEAD] = qt;  // pops that found the queue empty took fresh slots
        hi_c = min(S.ctl[C_HI], SC);
        over_c = S.ctl[C_OVERFLOW];
        t_next = next_event();
        __syncthreads();  // the reads above against phase X below
      }
      PHS_TICK(0)

      // ---- iterations: every own component whose next event lies inside the window processes it, at its own time
      while (t_next < wend && nrl_c - rl_base <= RLC / 2 && !over_c) {
        ++solve;
        ++iters;
        const int hi0 = hi_c;
        for (int s = tid; s < hi0; s += NT) {
          const double tcs = S.s_tc[s];
          if (!(tcs < wend)) continue;  // free slots hold +inf
          const int c = S.s_meta[s].z;
          const double tn = S.c_next[c];
          if (tcs > tn) continue;  // not the component's next event
          S.c_now[c] = tn;
          const uint4 pv = S.s_path[s];
          const bool activating = S.s_meta[s].y == -2;
          {  // the flow count of the path's links changes (a4 / a8)
            int nl = 0;
#pragma unroll
            for (int h = 0; h < kMaxHops; ++h) nl += path_at(pv, h) != (int)kNoLink;
            const int c0 = atomicAdd(&S.ctl[C_NCHG], nl);
            int k = 0;
#pragma unroll
            for (int h = 0; h < kMaxHops; ++h) {
              const int l = path_at(pv, h);
              if (l == (int)kNoLink) continue;
              atomicAdd(&S.l_n0[l], activating ? 1 : -1);
              S.l_chg[l] = solve;
              if (c0 + k < CLC) S.chg_list[c0 + k] = l;
              ++k;
            }
          }
          S.c_solve[c] = solve;
          if (activating) {  // PENDING -> ACTIVE
            S.s_rq[s] = -1;
            S.s_meta[s].y = -1;
            S.s_tc[s] = kInf;
            atomicAdd(&S.ctl[C_NACTIVE], 1);
            atomicSub(&S.ctl[C_NPEND], 1);
            continue;
          }
          // the flow completes at tn (bit-equal absolute time, S4.4): results, slot, successors (a8)
          const int f = S.s_meta[s].x;
          t_done[f] = tn;
          bneck_out[f] = S.l_gid[S.s_meta[s].y];
          const int nsucc = S.s_succ_cnt[s], sc0 = S.s_succ0[s], sc1 = S.s_succ1[s];
          S.s_meta[s].x = -1;
          S.s_tc[s] = kInf;
          atomicSub(&S.ctl[C_NACTIVE], 1);
          atomicAdd(&S.ctl[C_DONE], 1);
          S.free_q[atomicAdd(&S.ctl[C_QTAIL], 1) % SC] = s;
          // successors: one release-list entry each; counters and slots are handled at the end of the window (R)
          if (nsucc > 0) {
            const int i0 = atomicAdd(&S.ctl[C_NRL], nsucc);
            if (i0 + nsucc - rl_base > RLC) {
              S.ctl[C_OVERFLOW] = 1;
            } else {
              // t_act of a successor = max(start, LATEST predecessor) + Lat: every predecessor leaves its time
              const unsigned long long tb = (unsigned long long)__double_as_longlong(tn);
              if (nsucc <= 2) {
                S.rl_flow[i0 % RLC] = sc0;
                atomicMax(&t_rel[sc0], tb);
                if (nsucc > 1) {
                  S.rl_flow[(i0 + 1) % RLC] = sc1;
                  atomicMax(&t_rel[sc1], tb);
                }
              } else {
                for (int e = 0; e < nsucc; ++e) {
                  const int gs = succ[sc0 + e];
                  S.rl_flow[(i0 + e) % RLC] = gs;
                  atomicMax(&t_rel[gs], tb);
                }
              }
            }
          }
        }
        PHS_TICK(5)
        __syncthreads();
        PHS_TICK(6)
        const int nA = S.ctl[C_NACTIVE], nPend = S.ctl[C_NPEND];
        const int hi = hi_c = min(S.ctl[C_HI], SC);
        qtail_c = S.ctl[C_QTAIL];
        nrl_c = S.ctl[C_NRL];
        const int nchg = S.ctl[C_NCHG];
        over_c = S.ctl[C_OVERFLOW];
        max_active = max(max_active, nA);
        max_pending = max(max_pending, nPend);

        // ---- a5: fair share of the links whose flow count changed; components that had an event fold their next
        // event time again from their slots (F0, F)
        if (nchg <= CLC) {
          for (int i = tid; i < nchg; i += NT) {
            const int l = S.chg_list[i];
            const int n = S.l_n0[l];
            if (n > 0) S.l_share0[l] = fair_share(S.l_cap[l], n);  // a link listed twice is computed twice, alike
          }
        } else {  // the list overflowed: look at every link
          for (int l = tid; l < W.n_links; l += NT) {
            if (S.l_chg[l] != solve) continue;
            const int n = S.l_n0[l];
            if (n > 0) S.l_share0[l] = fair_share(S.l_cap[l], n);
          }
        }
        for (int c = tid; c < NCw; c += NT)
          if (S.c_solve[c] == solve) S.c_next[c] = kInf;
        __syncthreads();
        if (tid == 0) S.ctl[C_NCHG] = 0;  // read by everybody before the barrier above, written again in the next X
        PHS_TICK(7)

        // ---- rates (a6-a7): parallel progressive filling over the components this iteration touched
        auto freeze = [&](int s, int arg, long long rq, double tnow) {  // a7; R-LZ: only a changed rate touches the flow
          S.s_meta[s].y = arg;
          const long long old = S.s_rq[s];
          if (rq != old) {
            double rem = S.s_rem[s];
            if (old >= 0) {  // settle at the old rate: mul, sub, clamp
              rem = __dsub_rn(rem, __dmul_rn(rate_of(old), __dsub_rn(tnow, S.s_tl[s])));
              rem = rem > 0.0 ? rem : 0.0;
              S.s_rem[s] = rem;
            }
            S.s_tl[s] = tnow;
            S.s_rq[s] = rq;
            S.s_tc[s] = __dadd_rn(tnow, __ddiv_rn(rem, rate_of(rq)));  // S4.3: division, then addition
          }
        };
        int rounds = 1;
        ++g;
        for (int s = tid; s < hi; s += NT) {  // V0: arg-min link of every flow to re-solve (a6)
          const int4 m = S.s_meta[s];
          if (m.x < 0 || S.c_solve[m.z] != solve) continue;
          if (m.y == -2) {  // PENDING flow of a component that folds again
            smem_min_f64(&S.c_next[m.z], S.s_tc[s]);
            continue;
          }
          S.s_meta[s].y = -1;
          const uint4 pv = S.s_path[s];
          int p[kMaxHops];
          long long sh[kMaxHops];
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {
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
          for (int h = 0; h < kMaxHops; ++h) {
            const int l = p[h];
            if (l == (int)kNoLink) continue;
            if (l != arg) S.l_beat[l] = g;
            // working state of the solve's links (idempotent stores; debited from F0 on, after the barrier)
            S.l_caprem[l] = S.l_cap[l];
            S.l_nw[l] = S.l_n0[l];
            S.l_sharew[l] = sh[h];
          }
          S.s_meta[s].w = arg;
        }
        __syncthreads();
        bool left = false;
        for (int s = tid; s < hi; s += NT) {  // F0: unbeaten arg-min links freeze their flows and debit (a7), fold (a8)
          const int4 m = S.s_meta[s];
          if (m.x < 0 || m.y != -1) continue;  // only flows V0 opened are unfrozen here
          if (S.l_beat[m.w] != g) {
            const long long rq = S.l_share0[m.w];
            freeze(s, m.w, rq, S.c_now[m.z]);
            smem_min_f64(&S.c_next[m.z], S.s_tc[s]);
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
          } else {
            left = true;
          }
        }
        left = __syncthreads_or(left);
        PHS_TICK(8)
        if (left) {
          for (;;) {
            ++g;
            ++rounds;
            for (int s = tid; s < hi; s += NT) {  // V
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
            left = false;
            for (int s = tid; s < hi; s += NT) {  // F
              const int4 m = S.s_meta[s];
              if (m.x < 0 || m.y != -1) continue;
              const int arg = m.w;
              if (S.l_beat[arg] != g) {
                const long long rq = S.l_sharew[arg];
                freeze(s, arg, rq, S.c_now[m.z]);
                smem_min_f64(&S.c_next[m.z], S.s_tc[s]);
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
              } else {
                left = true;
              }
            }
            left = __syncthreads_or(left);
            if (!left) break;
          }
        }
        t_next = next_event();
        sum_active += nA;
        sum_rounds += rounds;
        PHS_TICK(9)
      }

      // ---- window end, barrier A: every CTA's release list is complete
      PHS_TICK(1)
      if (tid == 0) {
        mb.rl_base = rl_base;
        mb.rl_end = nrl_c;
      }
      cluster.sync();
      PHS_TICK(2)
      // ======== phase R (a8, DAG release): the flows released in this window become PENDING, in the CTA that owns
      // their component.  An entry is one predecessor's completion; the entry that brings the flow's counter to zero
      // creates the slot, with t_act = max(start, latest of the flow's predecessors) + Lat; the latest predecessor is
      // in the flow's word of t_rel (atomic max by every predecessor, ordered before this phase by barrier A).
      {
        const int qt = qtail_c;
        // the K lists as one index space: thread k fetches list k's bounds (one DSMEM trip for all of them)
        if (tid < K) {
          const Mailbox *o = cluster.map_shared_rank(&mb, tid);
          rl_lo[tid] = o->rl_base;
          rl_n[tid] = o->rl_end - o->rl_base;
        }
        __syncthreads();
        int total = 0;
        for (int k = 0; k < K; ++k) total += rl_n[k];
        for (int i = tid; i < total; i += NT) {
          int k = 0, j = i;
          while (j >= rl_n[k]) j -= rl_n[k++];
          const int gf = cluster.map_shared_rank(S.rl_flow, k)[(rl_lo[k] + j) % RLC];
          const unsigned cw = __ldcg(&fcw[gf]);
          if ((int)(cw >> 24) != me) continue;  // somebody else's flow
          // the record, the output position and the latest predecessor are fetched while the counter is in flight
          const FlowRec r = rec[gf];
          const int out = (int)fmap[gf];
          const double tr = __longlong_as_double((long long)__ldcg(&t_rel[gf]));
          if (atomicSub(&pred_cnt[gf], 1) != 1) continue;
          const double ta = __dadd_rn(r.start > tr ? r.start : tr, r.lat);
          const int h = atomicAdd(&S.ctl[C_QHEAD], 1);
          const int slot = h < qt ? S.free_q[h % SC] : atomicAdd(&S.ctl[C_HI], 1);
          if (slot >= SC) {
            S.ctl[C_OVERFLOW] = 1;
            continue;
          }
          atomicAdd(&S.ctl[C_NPEND], 1);
          fill_slot(slot, out, r, ta, (int)(cw & kLocMask));
          smem_min_f64(&S.c_next[cw & kLocMask], ta);
        }
        __syncthreads();
        rl_base = nrl_c;
        hi_c = min(S.ctl[C_HI], SC);
        t_next = next_event();
        if (tid == 0) {
          if (S.ctl[C_QHEAD] > qt) S.ctl[C_QHEAD] = qt;  // pops that found the queue empty took fresh slots
          mb.t_next = t_next;
          mb.live = S.ctl[C_NACTIVE] + S.ctl[C_NPEND];
          mb.over = S.ctl[C_OVERFLOW];
        }
      }
      PHS_TICK(3)
      cluster.sync();  // barrier B: lists consumed, post-R minima published
      PHS_TICK(4)
    }
#ifdef PHS_PHASE_CLOCKS
    if (tid == 0 && F > 100000)
      printf("unit %d cta %d/%d windows %d iters %d cycles: start %lld tail %lld barA %lld R %lld barB %lld | X %lld waitX %lld "
             "link %lld V0+F0 %lld rounds+fold %lld\n", inst, me, K, n_windows, iters, pc_[0], pc_[1], pc_[2], pc_[3], pc_[4],
             pc_[5], pc_[6], pc_[7], pc_[8], pc_[9]);
#endif

    // ---- results of the unit: CTA 0 adds up what the CTAs report
    if (tid == 0) {
      mb.done = S.ctl[C_DONE];
      mb.iters = iters;
      mb.sum_active = sum_active;
      mb.sum_rounds = sum_rounds;
      mb.max_active = max_active;
      mb.max_pending = max_pending;
      mb.max_slots = S.ctl[C_HI];
    }
    cluster.sync();
    if (me == 0 && tid == 0) {
      InstResult r;
      long long done = 0;
      r.n_events = 0; r.sum_active = 0; r.sum_par_rounds = 0; r.max_active = 0; r.max_pending = 0; r.max_slots = 0;
      for (int k = 0; k < K; ++k) {
        const Mailbox *o = cluster.map_shared_rank(&mb, k);
        done += o->done;
        if ((int64_t)o->iters > r.n_events) r.n_events = o->iters;  // the dependent chain: iterations of the busiest CTA
        r.sum_active += o->sum_active;
        r.sum_par_rounds += o->sum_rounds;
        r.max_active += o->max_active;
        r.max_pending += o->max_pending;
        r.max_slots = max(r.max_slots, o->max_slots);
      }
      r.status = status != PHS_OK ? status : (done < F ? PHS_ECYCLE : PHS_OK);
      r.path = 2;
      r.n_windows = n_windows;
      T.res[inst] = r;
    }
    cluster.sync();
  }
}

cudaError_t launch_window_path(const DevTables &t, const int32_t *list, int n, int *ticket, const WindowLaunch &w,
                               int n_clusters, cudaStream_t stream) {
  cudaError_t e = cudaFuncSetAttribute(phs_window_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(phs_window_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)w.smem);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute attr[1];
  cfg.gridDim = dim3((unsigned)(w.gang * n_clusters));
  cfg.blockDim = dim3(kWindowThreads);
  cfg.dynamicSmemBytes = w.smem;
  cfg.stream = stream;
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)w.gang;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, phs_window_kernel, t, list, n, ticket, w);
}

cudaError_t window_max_clusters(int gang, size_t smem, int *max_clusters) {
  cudaError_t e = cudaFuncSetAttribute(phs_window_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(phs_window_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute attr[1];
  cfg.gridDim = dim3((unsigned)gang);
  cfg.blockDim = dim3(kWindowThreads);
  cfg.dynamicSmemBytes = smem;
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)gang;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int n = 0;
  e = cudaOccupancyMaxActiveClusters(&n, phs_window_kernel, &cfg);
  if (e != cudaSuccess) {
    (void)cudaGetLastError();
    n = 0;
  }
  *max_clusters = n;
  return cudaSuccess;
}

}  // namespace phs
