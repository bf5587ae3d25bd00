// phs_kernels.cu -- CTA path of the hot path in CUDA for sm_100a: activation, max-min progressive filling (fair
// share per link, bottleneck argmin, freeze/scatter), event advance, retire + DAG release.
// a4-a9.  One CTA simulates one instance start to finish with ALL dynamic state in shared memory.
//
// Algorithm: the paper's water-filling freezes ONE bottleneck link per iteration (PAPER.md
// L165).  Because rates live on an exact integer grid (reading R-FX), freezing EVERY link whose (share, id) key is
// smaller than the key of every link it shares an unfrozen flow with ("local minimum") in one parallel round gives
// bit-identical rates, bottleneck ids and iteration count (proof in DESIGN.md).  A link is a local minimum iff every
// unfrozen flow on it names it as the arg-min link of its own path: count the votes per link and compare with the
// number of unfrozen flows on the link.  Phases of one event (barrier-separated):
//   X   advance all active flows to t_next, retire + release successors, activate what is due (a8, a4)
//   b0  first round: every flow computes the fair share of its own links (a5), votes for its arg-min (a6)
//   c   links holding all votes freeze their flows; debit paths; fold candidate completion times (a7, a8)
//   a,b later rounds: recompute the share of debited links (a5), vote again (a6)
#include <cuda_runtime.h>

#include <climits>

#include "phs_device.h"
#include "phs_devutil.cuh"

namespace phs {

namespace {

// ------------------------------------------------------------------------------------------------ smem layout
struct CtaSmem {
  long long *cap_rem, *share;      // [L]
  int *n, *nsnap, *cnt0, *cnt1;    // [L]
  int *leader;                     // [L] (event log only)
  unsigned char *dirty;            // [L]
  double *s_rem;                   // [S] remaining bytes
  long long *s_rq;                 // [S] rate in quanta
  int *s_flow, *s_bn, *s_arg;      // [S]
  int *s_path;                     // [S * kMaxHops]
  unsigned *s_succ_off;            // [S]
  int *s_succ_cnt, *s_succ0, *s_succ1;  // [S]
  int *free_q;                     // [S] FIFO of free slots
  double *p_time0, *p_time1;       // [S] pending lists (double buffered): activation time
  int *p_flow0, *p_flow1;          // [S]
  unsigned *pc8;                   // [(PCF+3)/4] predecessor counters, one byte per flow
  double *red;                     // [32] per-warp partial minima
  long long *red_key;              // [32] per-warp partial (share) for first_bneck
  int *red_id;                     // [32]
  int *ctl;                        // [32] control words
};
enum {
  C_HI = 0, C_QHEAD, C_QTAIL, C_NP0, C_NP1, C_NACTIVE, C_OVERFLOW, C_DONE, C_EV_NCOMP, C_EV_ROUNDS, C_EV_NACT0,
  C_EV_NACT1, C_NCTL
};

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

__host__ __device__ inline size_t carve(CtaSmem *s, unsigned char *base, int L, int S, int pcf, bool log) {
  size_t o = 0, a;
#define PHS_TAKE(field, type, count)                    \
  a = o;                                                \
  o = align_up(o + sizeof(type) * (size_t)(count), 16); \
  if (s) s->field = (type *)(base + a);
  PHS_TAKE(cap_rem, long long, L)
  PHS_TAKE(share, long long, L)
  PHS_TAKE(s_rem, double, S)
  PHS_TAKE(s_rq, long long, S)
  PHS_TAKE(p_time0, double, S)
  PHS_TAKE(p_time1, double, S)
  PHS_TAKE(red, double, 32)
  PHS_TAKE(red_key, long long, 32)
  PHS_TAKE(n, int, L)
  PHS_TAKE(nsnap, int, L)
  PHS_TAKE(cnt0, int, L)
  PHS_TAKE(cnt1, int, L)
  PHS_TAKE(leader, int, log ? L : 0)
  PHS_TAKE(s_flow, int, S)
  PHS_TAKE(s_bn, int, S)
  PHS_TAKE(s_arg, int, S)
  PHS_TAKE(s_path, int, S * kMaxHops)
  PHS_TAKE(s_succ_off, unsigned, S)
  PHS_TAKE(s_succ_cnt, int, S)
  PHS_TAKE(s_succ0, int, S)
  PHS_TAKE(s_succ1, int, S)
  PHS_TAKE(free_q, int, S)
  PHS_TAKE(p_flow0, int, S)
  PHS_TAKE(p_flow1, int, S)
  PHS_TAKE(pc8, unsigned, (pcf + 3) / 4)
  PHS_TAKE(red_id, int, 32)
  PHS_TAKE(ctl, int, 32)
  PHS_TAKE(dirty, unsigned char, L)
#undef PHS_TAKE
  return o;
}

}  // namespace

size_t cta_smem_bytes(int n_links, int slots, int pc_flows, bool log) {
  return carve(nullptr, nullptr, n_links, slots, pc_flows, log);
}

// ================================================================================================ CTA kernel
// NT threads; LOG: write the event log; PCS: predecessor counters live in shared memory (one byte per flow).
template <int NT, bool LOG, bool PCS>
__global__ void __launch_bounds__(NT) phs_cta_kernel(DevTables T, const int32_t *__restrict__ order, int n_order,
                                                     int *ticket, int SC, int pcf) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int sh_inst;
  CtaSmem S;
  const int L = T.n_links;
  carve(&S, smem_raw, L, SC, pcf, LOG);
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
    double *t_done = T.t_done + D.flow_base;
    int32_t *bneck_out = T.bneck + D.flow_base;
    const int64_t *__restrict__ capq = T.capq + (int64_t)inst * L;
    phs_event *log = (LOG && D.log_base >= 0) ? T.log + D.log_base : nullptr;
    const int F = D.n_flows;

    // ---- init: link state = full capacity, nothing active; flows without predecessors become PENDING (S4)
    for (int l = tid; l < L; l += NT) {
      S.cap_rem[l] = capq[l];
      S.n[l] = 0;
      S.cnt0[l] = 0;
      S.cnt1[l] = 0;
      if (LOG) S.leader[l] = INT_MAX;
      S.dirty[l] = 0;
    }
    for (int s = tid; s < SC; s += NT) {
      S.s_flow[s] = -1;
      S.s_bn[s] = -1;
    }
    if (tid < C_NCTL) S.ctl[tid] = 0;
    if (PCS) {
      const unsigned *src = (const unsigned *)(T.pred_cnt0_u8 + D.pc8_base);
      for (int w = tid; w < (F + 3) / 4; w += NT) S.pc8[w] = src[w];
    }
    __syncthreads();
    {
      const int32_t *__restrict__ pc0 = T.pred_cnt0 + D.flow_base;
      for (int f = tid; f < F; f += NT) {
        int pc;
        if (PCS) {
          pc = (S.pc8[f >> 2] >> ((f & 3) * 8)) & 0xff;
        } else {
          pc = pc0[f];
          pred_cnt[f] = pc;
        }
        if (pc == 0) {
          const double st = rec[f].start, la = rec[f].lat;
          const int i = atomicAdd(&S.ctl[C_NP0], 1);
          if (i < SC) {
            S.p_flow0[i] = f;
            S.p_time0[i] = __dadd_rn(st, la);
          } else {
            S.ctl[C_OVERFLOW] = 1;
          }
        }
      }
    }
    __syncthreads();

    double now = 0.0, t_next = 0.0;
    int cur = 0;   // which pending buffer is live
    int ev = -1;   // index of the event whose advance phase X is about to execute
    long long sum_active = 0, sum_rounds = 0;
    int max_active = 0, max_pending = 0;
    int status = PHS_OK;
    int first_bneck = -1;

    for (;;) {
      // ======== phase X (a8 + a4): advance to t_next, retire, release successors, activate what is due
      const double dt = __dsub_rn(t_next, now);
      const int hi0 = S.ctl[C_HI];
      const int qtail = S.ctl[C_QTAIL];
      const int nP = min(S.ctl[C_NP0 + cur], SC);
      int *const pf_cur = cur ? S.p_flow1 : S.p_flow0, *const pf_oth = cur ? S.p_flow0 : S.p_flow1;
      double *const pt_cur = cur ? S.p_time1 : S.p_time0, *const pt_oth = cur ? S.p_time0 : S.p_time1;
      int *const np_oth = &S.ctl[C_NP0 + (cur ^ 1)];
      double mymin = kInf;  // running min: pending activation times, and tc of my flows once frozen

      auto activate = [&](int f, const FlowRec &r) {
        const int h = atomicAdd(&S.ctl[C_QHEAD], 1);
        const int slot = h < qtail ? S.free_q[h % SC] : atomicAdd(&S.ctl[C_HI], 1);
        if (slot >= SC) {
          S.ctl[C_OVERFLOW] = 1;
          return;
        }
        S.s_flow[slot] = f;
        S.s_rem[slot] = r.bytes;
#pragma unroll
        for (int h2 = 0; h2 < kMaxHops; ++h2) {
          const int l = r.path[h2];
          if (l >= 0) atomicAdd(&S.n[l], 1);
          S.s_path[slot * kMaxHops + h2] = l;
        }
        S.s_succ_off[slot] = r.succ_off;
        S.s_succ_cnt[slot] = r.succ_cnt;
        S.s_succ0[slot] = r.succ_in[0];
        S.s_succ1[slot] = r.succ_in[1];
        atomicAdd(&S.ctl[C_NACTIVE], 1);
        if (LOG) atomicAdd(&S.ctl[C_EV_NACT0 + ((ev + 1) & 1)], 1);
      };
      auto release = [&](int g) {  // S4.5: pred_cnt--, at 0 -> t_act = max(start, now) + Lat
        bool zero;
        if (PCS) {
          const unsigned sh = (unsigned)(g & 3) * 8u;
          const unsigned old = atomicSub(&S.pc8[g >> 2], 1u << sh);
          zero = ((old >> sh) & 0xffu) == 1u;
        } else {
          zero = atomicSub(&pred_cnt[g], 1) == 1;
        }
        if (!zero) return;
        const FlowRec r = rec[g];
        const double ta = __dadd_rn(r.start > t_next ? r.start : t_next, r.lat);
        if (ta <= t_next) {
          activate(g, r);  // zero path latency: due at this very timestamp
        } else {
          const int i = atomicAdd(np_oth, 1);
          if (i < SC) {
            pf_oth[i] = g;
            pt_oth[i] = ta;
          } else {
            S.ctl[C_OVERFLOW] = 1;
          }
          mymin = dmin(mymin, ta);
        }
      };

      for (int s = tid; s < hi0; s += NT) {
        const int bn = S.s_bn[s];
        if (bn < 0) continue;  // free, or activated in this very phase
        const int f = S.s_flow[s];
        const long long rq = S.s_rq[s];
        const double rate = rate_of(rq);
        const double rem = S.s_rem[s];
        const double tc = __dadd_rn(now, __ddiv_rn(rem, rate));
        const bool done = tc == t_next;  // bit-equal absolute time (S4.4)
        S.cnt0[bn] = 0;
        S.cnt1[bn] = 0;
        if (LOG) S.leader[bn] = INT_MAX;
        S.s_bn[s] = -1;
        // undo the solve's debits (exact: integer arithmetic); survivors stay counted on their links
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {
          const int l = S.s_path[s * kMaxHops + h];
          if (l < 0) break;
          atomicAdd((unsigned long long *)&S.cap_rem[l], (unsigned long long)rq);
          if (!done) atomicAdd(&S.n[l], 1);
        }
        if (done) {
          t_done[f] = t_next;
          bneck_out[f] = bn;
          S.s_flow[s] = -1;
          S.free_q[atomicAdd(&S.ctl[C_QTAIL], 1) % SC] = s;
          atomicSub(&S.ctl[C_NACTIVE], 1);
          atomicAdd(&S.ctl[C_DONE], 1);
          if (LOG) atomicAdd(&S.ctl[C_EV_NCOMP], 1);
          const int nsucc = S.s_succ_cnt[s];
          if (nsucc > 0) release(S.s_succ0[s]);
          if (nsucc > 1) release(S.s_succ1[s]);
          if (nsucc > 2) {
            const unsigned e0 = S.s_succ_off[s];
            for (int e = 2; e < nsucc; ++e) release(succ[e0 + e]);
          }
        } else {
          const double r2 = __dsub_rn(rem, __dmul_rn(rate, dt));  // mul, then sub, then clamp
          S.s_rem[s] = r2 > 0.0 ? r2 : 0.0;
        }
      }
      for (int i = tid; i < nP; i += NT) {  // a4: PENDING flows whose activation time has come
        const int f = pf_cur[i];
        const double ta = pt_cur[i];
        if (ta <= t_next) {
          const FlowRec r = rec[f];
          activate(f, r);
        } else {
          const int j = atomicAdd(np_oth, 1);
          if (j < SC) {
            pf_oth[j] = f;
            pt_oth[j] = ta;
          } else {
            S.ctl[C_OVERFLOW] = 1;
          }
          mymin = dmin(mymin, ta);
        }
      }
      __syncthreads();
      now = t_next;
      if (tid == 0) {
        S.ctl[C_NP0 + cur] = 0;
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
      cur ^= 1;
      if (S.ctl[C_OVERFLOW]) {
        status = kOverflow;
        break;
      }
      const int nA = S.ctl[C_NACTIVE];
      const int nPend = S.ctl[C_NP0 + cur];
      if (nA == 0 && nPend == 0) break;  // S4.3: nothing active, nothing pending -> stop
      const int hi = S.ctl[C_HI];
      max_active = max(max_active, nA);
      max_pending = max(max_pending, nPend);

      // ======== rates: parallel progressive filling over the active set (a5-a7), tc folded in (a8)
      int round = 0;
      bool left = nA > 0;
      for (;;) {
        if (left) {
          int *cnt = (round & 1) ? S.cnt1 : S.cnt0;
          int *cnt_prev = (round & 1) ? S.cnt0 : S.cnt1;
          if (round > 0) {
            // (a) fair share of every link debited in the previous round
            for (int l = tid; l < L; l += NT) {
              if (S.dirty[l]) {
                S.dirty[l] = 0;
                const int nl = S.n[l];
                S.nsnap[l] = nl;
                if (nl > 0) S.share[l] = fair_share(S.cap_rem[l], nl);
              }
            }
            __syncthreads();
          }
          // (b) every unfrozen flow votes for the arg-min (share, id) link of its path.  In the first round the
          // flow computes the shares of its own links itself (cap_rem = capacity, n is final after phase X) and
          // publishes them, which saves the link pass and its barrier.
          long long bk = LLONG_MAX;
          int bl = INT_MAX;
          for (int s = tid; s < hi; s += NT) {
            if (S.s_flow[s] < 0 || S.s_bn[s] >= 0) continue;
            if (round > 0) cnt_prev[S.s_arg[s]] = 0;
            long long best = LLONG_MAX;
            int arg = -1;
#pragma unroll
            for (int h = 0; h < kMaxHops; ++h) {
              const int l = S.s_path[s * kMaxHops + h];
              if (l < 0) break;
              long long sh;
              if (round == 0) {
                const int nl = S.n[l];
                sh = fair_share(S.cap_rem[l], nl);
                S.share[l] = sh;
                S.nsnap[l] = nl;
              } else {
                sh = S.share[l];
              }
              if (sh < best || (sh == best && l < arg)) {
                best = sh;
                arg = l;
              }
            }
            S.s_arg[s] = arg;
            atomicAdd(&cnt[arg], 1);
            if (LOG) {
              atomicMin(&S.leader[arg], s);
              if (best < bk || (best == bk && arg < bl)) {
                bk = best;
                bl = arg;
              }
            }
          }
          if (LOG && round == 0) {  // O4 first_bneck = global arg-min = min over the flows' arg-mins
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
          __syncthreads();
          // (c) a link that collected the votes of ALL its unfrozen flows is a bottleneck: freeze them, debit paths
          bool mine_left = false;
          for (int s = tid; s < hi; s += NT) {
            if (S.s_flow[s] < 0 || S.s_bn[s] >= 0) continue;
            const int arg = S.s_arg[s];
            if (cnt[arg] == S.nsnap[arg]) {
              const long long rq = S.share[arg];
              S.s_rq[s] = rq;
              S.s_bn[s] = arg;
#pragma unroll
              for (int h = 0; h < kMaxHops; ++h) {
                const int l = S.s_path[s * kMaxHops + h];
                if (l < 0) break;
                atomicAdd((unsigned long long *)&S.cap_rem[l], (unsigned long long)(-rq));
                atomicSub(&S.n[l], 1);
                S.dirty[l] = 1;
              }
              // S4.3: candidate completion time, division then addition
              mymin = dmin(mymin, __dadd_rn(now, __ddiv_rn(S.s_rem[s], rate_of(rq))));
              if (LOG && S.leader[arg] == s) atomicAdd(&S.ctl[C_EV_ROUNDS], 1);
            } else {
              mine_left = true;
              if (LOG) S.leader[arg] = INT_MAX;
            }
          }
          left = mine_left;
          ++round;
        }
        const double wm = warp_min(mymin);
        if (lane == 0) S.red[warp] = wm;
        left = __syncthreads_or(left);
        if (!left) break;
      }
      // ======== next time (a8): t_next = min over candidate completion times and pending activations
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
      sum_rounds += round;
    }
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
      T.res[inst] = r;
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------ launchers
namespace {
template <int NT, bool LOG, bool PCS>
cudaError_t launch_one(const DevTables &t, const int32_t *order, int n, int *ticket, const CtaLaunch &c,
                       cudaStream_t stream) {
  cudaError_t e = cudaFuncSetAttribute(phs_cta_kernel<NT, LOG, PCS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)c.smem);
  if (e != cudaSuccess) return e;
  phs_cta_kernel<NT, LOG, PCS><<<c.grid, NT, c.smem, stream>>>(t, order, n, ticket, c.slots, c.pc_flows);
  return cudaGetLastError();
}
template <int NT>
cudaError_t launch_nt(const DevTables &t, const int32_t *order, int n, int *ticket, const CtaLaunch &c,
                      cudaStream_t stream) {
  const bool pcs = c.pc_flows > 0;
  if (c.log) return pcs ? launch_one<NT, true, true>(t, order, n, ticket, c, stream)
                        : launch_one<NT, true, false>(t, order, n, ticket, c, stream);
  return pcs ? launch_one<NT, false, true>(t, order, n, ticket, c, stream)
             : launch_one<NT, false, false>(t, order, n, ticket, c, stream);
}
}  // namespace

cudaError_t launch_cta_path(const DevTables &t, const int32_t *order, int n, int *ticket, const CtaLaunch &c,
                            cudaStream_t stream) {
  switch (c.threads) {
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
  for (int i = lane; i < n; i += 32) m = fmax(m, p[i]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  if (lane == 0) out[c] = m;
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
