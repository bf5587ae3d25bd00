// phs_cluster.cu -- cluster path of the hot path: one thread-block cluster (up to 16 CTAs, hardware cluster
// barrier) simulates one LARGE instance (SURVEY.md 8(a) a4-a9 for instances whose state does not fit one SM).
// Same algorithm as the CTA path (phs_kernels.cu): stamp-based local-minimum test, static-component re-solve, lazy
// settle (R-LZ).  What changes is where the state lives and how the CTAs combine:
//   * link state (32-byte LinkS + 16-byte LinkW per link) lives in global memory and stays L2-resident; it is read
//     with ld.cg and written with st.cg / atomics, because other SMs of the cluster write it;
//   * flow slots live in global memory too, but each CTA owns a private partition of the slot array (a flow is
//     created in the partition of the CTA that released it), so slot traffic is L1-cacheable and never contended;
//   * capacity debits are first summed per CTA in shared memory, then each touched link is debited once per CTA;
//   * per filling round: V (arg-min, beat stamps) | cluster barrier | F (freeze, settle, debit) + combine |
//     cluster barrier | R (shares of the debited links).
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include <climits>

#include "phs_device.h"
#include "phs_devutil.cuh"

namespace cg = cooperative_groups;

namespace phs {

namespace {

constexpr int NT = kClusterThreads;

// control block of one region, viewed as int[128] / unsigned long long[64]
enum {
  K_INST = 0, K_NACTIVE, K_NPEND, K_DONE, K_OVERFLOW, K_NCHG, K_NDL0, K_NDL1, K_LEFT0, K_LEFT1, K_LEFT2, K_EV_NACT0,
  K_EV_NACT1, K_EV_NCOMP, K_EV_ROUNDS, K_MAXSLOTS, K_FB_ID0 = 32 /* 16 per-CTA first_bneck ids */
};
constexpr int Q_TMIN0 = 24 /* [24],[25]: t_next minima by event parity */, Q_FB_KEY0 = 32 /* 16 per-CTA keys */;

// Per-CTA private flow slots.  Hot fields (read every round) live in shared memory; cold fields (touched when a
// flow's rate changes, or when it completes) live in a CTA-private partition of the region's global slot block.
struct Slots {
  // shared memory, 44 bytes per slot + two work lists
  double *tc;          // PENDING: activation time; ACTIVE: completion time; free: +inf
  long long *rq;       // rate in quanta, -1 before the first solve
  int *flow, *bn, *comp, *arg;
  unsigned short *path;  // [Sc * kMaxHops], kNoLink = none
  unsigned short *wl0, *wl1;
  // global memory
  double *rem, *tl;
  int *succ_cnt, *succ0, *succ1, *freeq;
};
constexpr unsigned short kNoLink = 0xffff;
constexpr int kSlotSmemBytes = 8 + 8 + 4 * 4 + 2 * kMaxHops + 2 * 2;  // 48

__host__ __device__ inline size_t slot_bytes_per_cta(int64_t Sc) {  // global part
  return ((size_t)Sc * (2 * 8 + 4 * 4) + 255) / 256 * 256;
}
__device__ inline void carve_slots(Slots &s, unsigned char *sm, unsigned char *gl, int64_t Sc) {
  s.tc = (double *)sm;
  s.rq = (long long *)(s.tc + Sc);
  s.flow = (int *)(s.rq + Sc);
  s.bn = s.flow + Sc;
  s.comp = s.bn + Sc;
  s.arg = s.comp + Sc;
  s.path = (unsigned short *)(s.arg + Sc);
  s.wl0 = s.path + Sc * kMaxHops;
  s.wl1 = s.wl0 + Sc;
  s.rem = (double *)gl;
  s.tl = s.rem + Sc;
  s.succ_cnt = (int *)(s.tl + Sc);
  s.succ0 = s.succ_cnt + Sc;
  s.succ1 = s.succ0 + Sc;
  s.freeq = s.succ1 + Sc;
}

// smem control words of a CTA
enum { M_HI = 0, M_QHEAD, M_QTAIL, M_DACT, M_DPEND, M_DDONE, M_NWL0, M_NWL1, M_NTOUCH, M_OVER, M_NCTL };

__device__ __forceinline__ void smem_add64(long long *p, long long v) {
  unsigned *w = (unsigned *)p;
  const unsigned lo = (unsigned)(unsigned long long)v, hi = (unsigned)((unsigned long long)v >> 32);
  const unsigned old = atomicAdd(w, lo);
  const unsigned carry = (old + lo) < old ? 1u : 0u;
  if (hi + carry) atomicAdd(w + 1, hi + carry);
}

__host__ __device__ inline size_t region_links_bytes(int L) {
  size_t o = (size_t)L * sizeof(LinkS) + (size_t)L * sizeof(LinkW) + (size_t)L * 4 * 2;  // + solve, won
  return (o + 255) / 256 * 256;
}

}  // namespace

size_t cluster_region_bytes(int L, int64_t Sc, int cluster_size) {
  return region_links_bytes(L) + 512 + (size_t)cluster_size * slot_bytes_per_cta(Sc);
}
size_t cluster_smem_bytes(int L, int64_t Sc, bool aggregate) {
  return (aggregate ? (size_t)L * 16 : 16) + (size_t)Sc * kSlotSmemBytes + 16;
}

// ================================================================================================ cluster kernel
// LOG: write the event log (and solve every component at every event); AGG: debits are pre-summed in shared memory.
template <bool LOG, bool AGG>
__global__ void __launch_bounds__(kClusterThreads, 1)
    phs_cluster_kernel(DevTables T, const int32_t *__restrict__ list, int n_list, int *ticket, ClusterScratch SC) {
  cg::cluster_group cluster = cg::this_cluster();
  const int CS = (int)cluster.num_blocks();
  const int crank = (int)cluster.block_rank();
  const int region = blockIdx.x / CS;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int ctid = crank * NT + tid;  // thread index within the cluster
  const int CT = CS * NT;             // threads in the cluster
  const int L = T.n_links;
  const int Sc = (int)SC.Sc;

  // ---- carve this cluster's region
  unsigned char *rb = SC.base + (size_t)region * SC.region_bytes;
  LinkS *LS = (LinkS *)rb;
  LinkW *LW = (LinkW *)(LS + L);
  int *solve_g = (int *)(LW + L);
  int *won = solve_g + L;
  unsigned long long *ctrl64 = (unsigned long long *)(rb + region_links_bytes(L));
  int *ctl_g = (int *)ctrl64;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  long long *dcap_loc = (long long *)smem_raw;  // [L]   (AGG)
  int *dn_loc = (int *)(dcap_loc + L);          // [L]
  int *touched = dn_loc + L;                    // [L]
  Slots S;
  carve_slots(S, smem_raw + (AGG ? (size_t)L * 16 : 16),
              rb + region_links_bytes(L) + 512 + (size_t)crank * slot_bytes_per_cta(Sc), Sc);
  __shared__ double red[32];
  __shared__ long long red_key[32];
  __shared__ int red_id[32];
  __shared__ int ctl[M_NCTL];

  for (;;) {
    // ---- a9: clusters pull instances from the list
    if (ctid == 0) __stcg(&ctl_g[K_INST], atomicAdd(ticket, 1));
    cluster.sync();
    const int qi = __ldcg(&ctl_g[K_INST]);
    cluster.sync();
    if (qi >= n_list) break;
    const int inst = list[qi];
    const InstDesc D = T.inst[inst];
    const FlowRec *__restrict__ rec = T.rec + D.flow_base;
    const int32_t *__restrict__ succ = T.succ + D.succ_base;
    const int32_t *__restrict__ pc0 = T.pred_cnt0 + D.flow_base;
    int32_t *pred_cnt = T.pred_cnt + D.flow_base;
    double *t_done = T.t_done + D.flow_base;
    int32_t *bneck_out = T.bneck + D.flow_base;
    const int64_t *__restrict__ capq = T.capq + (int64_t)inst * L;
    const int32_t *__restrict__ lcomp = T.lcomp + (int64_t)inst * L;
    phs_event *log = (LOG && D.log_base >= 0) ? T.log + D.log_base : nullptr;
    const int F = D.n_flows;

    // ---- init: no flow anywhere, every slot free
    for (int l = ctid; l < L; l += CT) {
      LinkS z;
      z.share0 = 0; z.sharew = 0; z.wsolve = 0; z.n0 = 0; z.beat = 0; z.chg = 0;
      LS[l] = z;
      LinkW w;
      w.caprem = 0; w.nw = 0; w.deb = 0;
      LW[l] = w;
      solve_g[l] = 0;
      won[l] = 0;
    }
    if (ctid >= 1 && ctid < 128) ctl_g[ctid] = 0;
    for (int s = tid; s < Sc; s += NT) {
      S.flow[s] = -1;
      S.tc[s] = kInf;
    }
    if (tid < M_NCTL) ctl[tid] = 0;
    if (AGG)
      for (int l = tid; l < L; l += NT) {
        dcap_loc[l] = 0;
        dn_loc[l] = 0;
      }
    cluster.sync();
    if (ctid == 0) {
      ctrl64[Q_TMIN0] = (unsigned long long)__double_as_longlong(kInf);
      ctrl64[Q_TMIN0 + 1] = (unsigned long long)__double_as_longlong(kInf);
    }

    auto fill_slot = [&](int slot, int f, const FlowRec &r, double ta) {
      S.flow[slot] = f;
      S.rem[slot] = r.bytes;
      S.bn[slot] = -2;
      S.comp[slot] = r.comp;
#pragma unroll
      for (int h = 0; h < kMaxHops; ++h)
        S.path[slot * kMaxHops + h] = r.path[h] < 0 ? kNoLink : (unsigned short)r.path[h];
      S.succ_cnt[slot] = r.succ_cnt;
      S.succ0[slot] = r.succ_in[0];
      S.succ1[slot] = r.succ_in[1];
      S.tc[slot] = ta;
    };

    // S4: flows without predecessors become PENDING; flow f starts in the partition of CTA f mod CS
    for (int64_t f = crank + (int64_t)CS * tid; f < F; f += (int64_t)CS * NT) {
      const int pc = pc0[f];
      pred_cnt[f] = pc;
      if (pc == 0) {
        const FlowRec r = rec[f];
        const int slot = atomicAdd(&ctl[M_HI], 1);
        if (slot < Sc) {
          fill_slot(slot, (int)f, r, __dadd_rn(r.start, r.lat));
          atomicAdd(&ctl[M_DPEND], 1);
        } else {
          ctl[M_OVER] = 1;
        }
      }
    }
    __syncthreads();
    if (tid == 0) {
      if (ctl[M_DPEND]) atomicAdd(&ctl_g[K_NPEND], ctl[M_DPEND]);
      ctl[M_DPEND] = 0;
      if (ctl[M_OVER]) __stcg(&ctl_g[K_OVERFLOW], 1);
    }
    cluster.sync();

    double now = 0.0, t_next = 0.0;
    int ev = -1, solve = 0, g = 0, it = 0;
    long long sum_active = 0, sum_rounds = 0;
    int max_active = 0, max_pending = 0;
    int status = PHS_OK;
    int first_bneck = -1;

    for (;;) {
      // ======== phase X (a8 + a4): retire what completes at t_next, release successors, activate what is due
      ++solve;
      const int hi0 = min(ctl[M_HI], Sc);
      const int qtail = ctl[M_QTAIL];
      auto touch_link = [&](int l, int delta) {  // the link's flow count changes: its share0 is stale for this
        atomicAdd(&LS[l].n0, delta);             // event's solve (no value returns: both are fire-and-forget)
        __stcg(&LS[l].chg, solve);
      };
      auto activate = [&](int slot) {
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {
          const int l = S.path[slot * kMaxHops + h];
          if (l == kNoLink) break;
          touch_link(l, 1);
        }
        __stcg(&solve_g[S.comp[slot]], solve);
        S.rq[slot] = -1;
        S.bn[slot] = -1;
        S.tc[slot] = kInf;
        atomicAdd(&ctl[M_DACT], 1);
        atomicSub(&ctl[M_DPEND], 1);
      };
      auto make_pending = [&](int gf, const FlowRec &r) {  // S4.5: t_act = max(start, now) + Lat
        const double ta = __dadd_rn(r.start > t_next ? r.start : t_next, r.lat);
        const int h = atomicAdd(&ctl[M_QHEAD], 1);
        const int slot = h < qtail ? S.freeq[h % Sc] : atomicAdd(&ctl[M_HI], 1);
        if (slot >= Sc) {
          ctl[M_OVER] = 1;
          return;
        }
        atomicAdd(&ctl[M_DPEND], 1);
        const bool due = ta <= t_next;
        fill_slot(slot, gf, r, due ? kInf : ta);
        if (due) activate(slot);
      };
      auto release = [&](int gf) {
        if (atomicSub(&pred_cnt[gf], 1) != 1) return;
        const FlowRec r = rec[gf];
        make_pending(gf, r);
      };
      auto release2 = [&](int g0, int g1) {  // both counters, then both records: the round trips overlap
        const bool z0 = g0 >= 0 && atomicSub(&pred_cnt[g0], 1) == 1;
        const bool z1 = g1 >= 0 && atomicSub(&pred_cnt[g1], 1) == 1;
        FlowRec r0, r1;
        if (z0) r0 = rec[g0];
        if (z1) r1 = rec[g1];
        if (z0) make_pending(g0, r0);
        if (z1) make_pending(g1, r1);
      };
      for (int s = tid; s < hi0; s += NT) {
        if (!(S.tc[s] <= t_next)) continue;
        if (S.bn[s] == -2) {
          activate(s);
          continue;
        }
        const int f = S.flow[s];
        t_done[f] = t_next;
        bneck_out[f] = S.bn[s];
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {
          const int l = S.path[s * kMaxHops + h];
          if (l == kNoLink) break;
          touch_link(l, -1);
        }
        __stcg(&solve_g[S.comp[s]], solve);
        S.flow[s] = -1;
        S.tc[s] = kInf;
        S.freeq[atomicAdd(&ctl[M_QTAIL], 1) % Sc] = s;
        atomicSub(&ctl[M_DACT], 1);
        atomicAdd(&ctl[M_DDONE], 1);
        const int nsucc = S.succ_cnt[s];
        if (nsucc <= 2) {
          if (nsucc > 0) release2(S.succ0[s], nsucc > 1 ? S.succ1[s] : -1);
        } else {
          const int e0 = S.succ0[s];
          for (int e = 0; e < nsucc; ++e) release(succ[e0 + e]);
        }
      }
      __syncthreads();
      if (tid == 0) {  // this CTA's net changes of the cluster-wide counters
        const int dact = ctl[M_DACT], dpend = ctl[M_DPEND], ddone = ctl[M_DDONE];
        if (dact) atomicAdd(&ctl_g[K_NACTIVE], dact);
        if (dpend) atomicAdd(&ctl_g[K_NPEND], dpend);
        if (ddone) atomicAdd(&ctl_g[K_DONE], ddone);
        if (LOG) {
          if (ddone) atomicAdd(&ctl_g[K_EV_NCOMP], ddone);
          if (dact + ddone) atomicAdd(&ctl_g[K_EV_NACT0 + ((ev + 1) & 1)], dact + ddone);  // activations
        }
        ctl[M_DACT] = 0;
        ctl[M_DPEND] = 0;
        ctl[M_DDONE] = 0;
        if (ctl[M_QHEAD] > qtail) ctl[M_QHEAD] = qtail;
        if (ctl[M_OVER]) __stcg(&ctl_g[K_OVERFLOW], 1);
        atomicMax(&ctl_g[K_MAXSLOTS], ctl[M_HI]);
        ctl[M_NWL0] = 0;
        ctl[M_NWL1] = 0;
      }
      cluster.sync();  // ---------------------------------------------------------------- cluster barrier X
      now = t_next;
      const int nA = __ldcg(&ctl_g[K_NACTIVE]);
      const int nPend = __ldcg(&ctl_g[K_NPEND]);
      if (LOG && ctid == 0) {
        if (log && ev >= 0) {  // O4: the event that just finished
          phs_event e;
          e.t = now;
          e.n_completed = __ldcg(&ctl_g[K_EV_NCOMP]);
          e.n_activated = __ldcg(&ctl_g[K_EV_NACT0 + (ev & 1)]);
          e.n_rounds = __ldcg(&ctl_g[K_EV_ROUNDS]);
          e.first_bneck = first_bneck;
          log[ev] = e;
        }
        __stcg(&ctl_g[K_EV_NCOMP], 0);
        __stcg(&ctl_g[K_EV_ROUNDS], 0);
        if (ev >= 0) __stcg(&ctl_g[K_EV_NACT0 + (ev & 1)], 0);
      }
      ++ev;
      if (__ldcg(&ctl_g[K_OVERFLOW])) {
        status = kOverflow;
        break;
      }
      if (nA == 0 && nPend == 0) break;
      const int hi = min(ctl[M_HI], Sc);
      max_active = max(max_active, nA);
      max_pending = max(max_pending, nPend);
      const int par = ev & 1;

      // ======== P: working capacities of the links that will be re-solved (split over the cluster; they are first
      // debited after cluster barrier 1)
      for (int l = ctid; l < L; l += CT) {
        if (LOG || __ldcg(&solve_g[__ldg(&lcomp[l])]) == solve) {
          __stcg(&LW[l].caprem, (long long)__ldg(&capq[l]));
          __stcg(&LW[l].nw, __ldcg(&LS[l].n0));
        }
      }
      // ======== rates (a5-a7): parallel progressive filling over the components this event touched
      unsigned short *wl = S.wl0, *wl_next = S.wl1;
      int nwl_idx = M_NWL0;
      double mymin = kInf;  // completion / activation times of this thread's flows, folded as they become final
      // a5 + a6: the fair share of every link of the flow's path, refreshed by the flow itself where it is stale
      // (every flow on such a link computes and stores the same value), arg-min (share, id), beat the other links
      auto vote = [&](int s, bool first) {
        int p[kMaxHops], pb[kMaxHops];
        long long sh[kMaxHops];
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {  // all loads first: one L2 round trip for the whole path
          const int l = p[h] = S.path[s * kMaxHops + h];
          sh[h] = LLONG_MAX;
          pb[h] = g;
          if (l == kNoLink) continue;
          const longlong2 a = __ldcg((const longlong2 *)&LS[l]);
          const int4 b = __ldcg((const int4 *)&LS[l] + 1);
          pb[h] = b.z;
          if (first) {
            if (b.w == solve) {  // flow count changed in this event
              sh[h] = fair_share(__ldg(&capq[l]), b.y);
              __stcg(&LS[l].share0, sh[h]);
            } else {
              sh[h] = a.x;
            }
          } else {
            const longlong2 w = __ldcg((const longlong2 *)&LW[l]);
            if ((int)(w.y >> 32) == g - 1) {  // debited in the previous round
              sh[h] = fair_share(w.x, (int)(unsigned)(unsigned long long)w.y);
              __stcg(&LS[l].sharew, sh[h]);
              __stcg(&LS[l].wsolve, solve);
            } else {
              sh[h] = b.x == solve ? a.y : a.x;
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
          if (p[h] != kNoLink && p[h] != arg && pb[h] != g) __stcg(&LS[p[h]].beat, g);
        S.arg[s] = arg;
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
          S.tc[s] = __dadd_rn(now, __ddiv_rn(rem, rate_of(rq)));
        }
        mymin = dmin(mymin, S.tc[s]);
        if (LOG && atomicExch(&won[arg], g) != g) atomicAdd(&ctl_g[K_EV_ROUNDS], 1);
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {  // debit the path
          const int l = S.path[s * kMaxHops + h];
          if (l == kNoLink) break;
          if (AGG) {
            if (atomicAdd(&dn_loc[l], 1) == 0) touched[atomicAdd(&ctl[M_NTOUCH], 1)] = l;
            smem_add64(&dcap_loc[l], rq);
          } else {
            atomicAdd((unsigned long long *)&LW[l].caprem, (unsigned long long)(-rq));
            atomicSub(&LW[l].nw, 1);
            __stcg(&LW[l].deb, g);
          }
        }
      };

      int rounds = 0;
      ++g;
      {  // ---- V0: collect the flows to re-solve, vote; fold the times of everybody else
        long long bk = LLONG_MAX;
        int bl = INT_MAX;
        for (int s = tid; s < hi; s += NT) {
          if (S.flow[s] < 0) continue;
          const bool in = S.bn[s] != -2 && (LOG || __ldcg(&solve_g[S.comp[s]]) == solve);
          if (!in) {
            mymin = dmin(mymin, S.tc[s]);
            continue;
          }
          S.bn[s] = -1;
          const longlong2 v = vote(s, true);
          wl[atomicAdd(&ctl[nwl_idx], 1)] = (unsigned short)s;
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
            __stcg((long long *)&ctrl64[Q_FB_KEY0 + crank], bk);
            __stcg(&ctl_g[K_FB_ID0 + crank], bl);
          }
        }
      }
      for (;;) {
        cluster.sync();  // -------------------------------------------------------------- cluster barrier 1
        if (rounds == 0 && ctid == 0) {  // everybody has read these for this event
          __stcg((long long *)&ctrl64[Q_TMIN0 + (par ^ 1)], __double_as_longlong(kInf));
        }
        ++rounds;
        // ---- F: flows whose arg-min link is unbeaten freeze (a7), settle (R-LZ) and debit; the rest stay listed
        const int nwl = ctl[nwl_idx];
        const int nxt_idx = nwl_idx == M_NWL0 ? M_NWL1 : M_NWL0;
        bool left = false;
        for (int i = tid; i < nwl; i += NT) {
          const int s = wl[i];
          const int arg = S.arg[s];
          const longlong2 a = __ldcg((const longlong2 *)&LS[arg]);
          const int4 b = __ldcg((const int4 *)&LS[arg] + 1);
          if (b.z != g) {
            freeze(s, arg, (rounds > 1 && b.x == solve) ? a.y : a.x);
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
            atomicAdd((unsigned long long *)&LW[l].caprem, (unsigned long long)(-dcap_loc[l]));
            atomicSub(&LW[l].nw, dn_loc[l]);
            __stcg(&LW[l].deb, g);
            dcap_loc[l] = 0;
            dn_loc[l] = 0;
          }
        }
        if (warp == 0) {
          const double m = warp_min(lane < NT / 32 ? red[lane] : kInf);
          if (lane == 0) atomicMin(&ctrl64[Q_TMIN0 + par], (unsigned long long)__double_as_longlong(m));
        }
        if (tid == 0) {
          if (left) __stcg(&ctl_g[K_LEFT0 + it % 3], 1);
          if (crank == 0) __stcg(&ctl_g[K_LEFT0 + (it + 2) % 3], 0);  // last read two barriers ago
        }
        mymin = kInf;  // folded
        cluster.sync();  // -------------------------------------------------------------- cluster barrier 2
        if (tid == 0) {  // everybody has consumed this round's lists
          ctl[nwl_idx] = 0;
          ctl[M_NTOUCH] = 0;
        }
        const bool any_left = __ldcg(&ctl_g[K_LEFT0 + it % 3]) != 0;
        ++it;
        if (!any_left) break;
        __syncthreads();
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
      t_next = __longlong_as_double((long long)__ldcg(&ctrl64[Q_TMIN0 + par]));
      if (LOG && ctid == 0) {
        first_bneck = -1;
        if (nA > 0) {
          long long bk = LLONG_MAX;
          for (int c = 0; c < CS; ++c) {
            const long long k = (long long)__ldcg(&ctrl64[Q_FB_KEY0 + c]);
            const int id = __ldcg(&ctl_g[K_FB_ID0 + c]);
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
    if (ctid == 0) {
      InstResult r;
      r.status = status != PHS_OK ? status : (__ldcg(&ctl_g[K_DONE]) < F ? PHS_ECYCLE : PHS_OK);
      r.path = 1;
      r.n_events = ev;
      r.sum_active = sum_active;
      r.sum_par_rounds = sum_rounds;
      r.max_active = max_active;
      r.max_pending = max_pending;
      r.max_slots = __ldcg(&ctl_g[K_MAXSLOTS]);
      r.pad_ = 0;
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
  const size_t smem = cluster_smem_bytes(t.n_links, s.Sc, AGG);
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

cudaError_t cluster_path_limits(int want, size_t smem, int *cluster_size, int *max_clusters) {
  cudaError_t e = prepare<true, true>(smem);
  if (e != cudaSuccess) return e;
  for (int cs = want; cs >= 1; cs >>= 1) {
    cudaLaunchConfig_t cfg{};
    cudaLaunchAttribute attr[1];
    set_cluster_attr(cfg, attr, cs, 1, smem, nullptr);
    int n = 0;
    e = cudaOccupancyMaxActiveClusters(&n, phs_cluster_kernel<true, true>, &cfg);
    if (e == cudaSuccess && n >= 1) {
      *cluster_size = cs;
      *max_clusters = n;
      return cudaSuccess;
    }
  }
  (void)cudaGetLastError();
  return cudaErrorLaunchOutOfResources;
}

}  // namespace phs
