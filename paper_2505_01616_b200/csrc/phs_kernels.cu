// phs_kernels.cu -- the hot path in CUDA for sm_100a: activation, max-min progressive filling (fair-share per
// link, bottleneck argmin, freeze/scatter), event advance, retire + DAG release.  SURVEY.md sec 8(a) rows a4-a9.
//
// Algorithm: the paper's water-filling freezes ONE bottleneck link per iteration (PAPER.md
// L165).  Because rates live on an exact integer grid (reading R-FX), freezing EVERY link whose (share, id) key is
// smaller than the key of every link it shares an unfrozen flow with ("local minimum") in one parallel round gives
// bit-identical rates, bottleneck ids and iteration count (proof in DESIGN.md).  A link is a local minimum iff every
// unfrozen flow on it names it as the arg-min link of its own path: count the votes per link and compare with the
// number of unfrozen flows on the link.  Each round is three barrier-separated phases:
//   (a) per dirty link:    share = cap_rem / n                 (fair-share segmented reduction; a5)
//   (b) per unfrozen flow: arg-min (share, link id) over its path, vote            (bottleneck argmin; a6)
//   (c) per unfrozen flow: if its arg link collected all votes -> freeze at share, debit the path   (a7)
// and the candidate completion time of a flow is folded into a running minimum as soon as it is frozen (a8).
#include <cuda_runtime.h>

#include <climits>

#include "phs_device.h"
#include "phs_devutil.cuh"

namespace phs {

namespace {

// ------------------------------------------------------------------------------------------------ smem layout
struct CtaSmem {
  long long *cap_rem, *share;  // [L]
  int *n, *nsnap, *cnt0, *cnt1, *leader;  // [L]
  unsigned char *dirty;        // [L]
  double *s_rem;               // [ACAP]
  long long *s_rq;             // [ACAP]
  int *s_flow, *s_bn, *s_arg;  // [ACAP]
  int *s_path;                 // [ACAP * kMaxHops]
  int *free_stack;             // [ACAP]
  double *p_tact0, *p_tact1;   // [PCAP] pending lists, double buffered
  int *p_flow0, *p_flow1;      // [PCAP]
  double *red;                 // [32] per-warp partial minima
  long long *red_key;          // [32] per-warp partial (share) for first_bneck
  int *red_id;                 // [32]
  int *ctl;                    // [16] control words
};
enum { C_HI = 0, C_NFREE, C_NP0, C_NP1, C_NACTIVE, C_OVERFLOW, C_EV_NACT, C_EV_NCOMP, C_EV_ROUNDS, C_DONE, C_NCTL };

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

__host__ __device__ inline size_t carve(CtaSmem *s, unsigned char *base, int L, int acap, int pcap) {
  size_t o = 0;
  auto take = [&](size_t bytes) {
    size_t at = o;
    o = align_up(o + bytes, 16);
    return at;
  };
  size_t a;
#define PHS_TAKE(field, type, count)        \
  a = take(sizeof(type) * (size_t)(count)); \
  if (s) s->field = (type *)(base + a);
  PHS_TAKE(cap_rem, long long, L)
  PHS_TAKE(share, long long, L)
  PHS_TAKE(s_rem, double, acap)
  PHS_TAKE(s_rq, long long, acap)
  PHS_TAKE(p_tact0, double, pcap)
  PHS_TAKE(p_tact1, double, pcap)
  PHS_TAKE(red, double, 32)
  PHS_TAKE(red_key, long long, 32)
  PHS_TAKE(n, int, L)
  PHS_TAKE(nsnap, int, L)
  PHS_TAKE(cnt0, int, L)
  PHS_TAKE(cnt1, int, L)
  PHS_TAKE(leader, int, L)
  PHS_TAKE(s_flow, int, acap)
  PHS_TAKE(s_bn, int, acap)
  PHS_TAKE(s_arg, int, acap)
  PHS_TAKE(s_path, int, acap * kMaxHops)
  PHS_TAKE(free_stack, int, acap)
  PHS_TAKE(p_flow0, int, pcap)
  PHS_TAKE(p_flow1, int, pcap)
  PHS_TAKE(red_id, int, 32)
  PHS_TAKE(ctl, int, 16)
  PHS_TAKE(dirty, unsigned char, L)
#undef PHS_TAKE
  return o;
}

}  // namespace

size_t cta_smem_bytes(int n_links, int acap, int pcap) { return carve(nullptr, nullptr, n_links, acap, pcap); }

// ================================================================================================ CTA path
// One CTA simulates one instance start to finish; link state, the active set and the pending list live in
// shared memory, per-flow records are gathered from global memory (L2) once per activation / release.
template <int NT, bool LOG>
__global__ void __launch_bounds__(NT) phs_cta_kernel(DevTables T, const int32_t *__restrict__ order, int n_order,
                                                     int *ticket, int acap, int pcap) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int sh_inst;
  CtaSmem S;
  const int L = T.n_links;
  carve(&S, smem_raw, L, acap, pcap);
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
    const FlowRec *__restrict__ rec = T.rec + D.rec_base;
    const int32_t *__restrict__ path = T.path + D.path_base;
    const int32_t *__restrict__ succ = T.succ + D.succ_base;
    const int32_t *__restrict__ pc0 = T.pred_cnt0 + D.flow_base;
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
      S.leader[l] = INT_MAX;
      S.dirty[l] = 0;
    }
    if (tid < C_NCTL) S.ctl[tid] = 0;
    __syncthreads();
    for (int f = tid; f < F; f += NT) {
      const int pc = pc0[f];
      pred_cnt[f] = pc;
      if (pc == 0) {
        const FlowRec r = rec[f];
        const int i = atomicAdd(&S.ctl[C_NP0], 1);
        if (i < pcap) {
          S.p_flow0[i] = f;
          S.p_tact0[i] = __dadd_rn(r.start, r.lat);
        } else {
          S.ctl[C_OVERFLOW] = 1;
        }
      }
    }
    __syncthreads();

    double now = 0.0;
    int cur = 0;  // which pending buffer is live
    long long n_events = 0, sum_active = 0, sum_rounds = 0;
    int max_active = 0, max_pending = 0;
    int status = PHS_OK;

    for (;;) {
      // ======== P0 (a4): activate PENDING flows with t_act <= now; survivors move to the other buffer
      // (an overflowing pending counter is clamped here and reported right after the barrier below)
      const int nP = min(S.ctl[C_NP0 + cur], pcap);
      int *const pf_cur = cur ? S.p_flow1 : S.p_flow0, *const pf_oth = cur ? S.p_flow0 : S.p_flow1;
      double *const pt_cur = cur ? S.p_tact1 : S.p_tact0, *const pt_oth = cur ? S.p_tact0 : S.p_tact1;
      double mymin = kInf;  // running min over: pending t_act, and tc of my flows once frozen
      for (int i = tid; i < nP; i += NT) {
        const int f = pf_cur[i];
        const double ta = pt_cur[i];
        if (ta <= now) {
          int slot;
          const int k = atomicSub(&S.ctl[C_NFREE], 1) - 1;
          if (k >= 0)
            slot = S.free_stack[k];
          else
            slot = atomicAdd(&S.ctl[C_HI], 1);
          if (slot < acap) {
            const FlowRec r = rec[f];
            const uint32_t pe = rec[f + 1].path_off;
            S.s_flow[slot] = f;
            S.s_rem[slot] = r.bytes;
            S.s_bn[slot] = -1;
#pragma unroll
            for (int h = 0; h < kMaxHops; ++h) {
              int l = -1;
              if (r.path_off + h < pe) {
                l = path[r.path_off + h];
                atomicAdd(&S.n[l], 1);
                S.dirty[l] = 1;
              }
              S.s_path[slot * kMaxHops + h] = l;
            }
            atomicAdd(&S.ctl[C_NACTIVE], 1);
            if (LOG) atomicAdd(&S.ctl[C_EV_NACT], 1);
          } else {
            S.ctl[C_OVERFLOW] = 1;
          }
        } else {
          const int j = atomicAdd(&S.ctl[C_NP0 + (cur ^ 1)], 1);  // < pcap: at most nP survivors
          pf_oth[j] = f;
          pt_oth[j] = ta;
          mymin = dmin(mymin, ta);
        }
      }
      __syncthreads();
      if (tid == 0) {
        S.ctl[C_NP0 + cur] = 0;
        if (S.ctl[C_NFREE] < 0) S.ctl[C_NFREE] = 0;
        if (LOG) {  // completions / frozen links of the previous event are final now: patch its log row
          if (log && n_events > 0) {
            log[n_events - 1].n_completed = S.ctl[C_EV_NCOMP];
            log[n_events - 1].n_rounds = S.ctl[C_EV_ROUNDS];
          }
          S.ctl[C_EV_NCOMP] = 0;
          S.ctl[C_EV_ROUNDS] = 0;
        }
      }
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
          // (a) fair share of every link whose (cap_rem, n) changed
          long long bk = LLONG_MAX;
          int bl = INT_MAX;
          for (int l = tid; l < L; l += NT) {
            if (S.dirty[l]) {
              S.dirty[l] = 0;
              const int nl = S.n[l];
              S.nsnap[l] = nl;
              if (nl > 0) S.share[l] = fair_share(S.cap_rem[l], nl);
            }
            if (LOG && round == 0 && S.n[l] > 0) {
              const long long sh = S.share[l];
              if (sh < bk) {  // ascending l: strict < keeps the lowest id among ties
                bk = sh;
                bl = l;
              }
            }
          }
          if (LOG && round == 0) {
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
          // (b) every unfrozen flow votes for the arg-min link of its path
          for (int s = tid; s < hi; s += NT) {
            if (S.s_flow[s] < 0 || S.s_bn[s] >= 0) continue;
            if (round > 0) cnt_prev[S.s_arg[s]] = 0;
            long long best = LLONG_MAX;
            int arg = -1;
#pragma unroll
            for (int h = 0; h < kMaxHops; ++h) {
              const int l = S.s_path[s * kMaxHops + h];
              if (l < 0) break;
              const long long sh = S.share[l];
              if (sh < best || (sh == best && l < arg)) {
                best = sh;
                arg = l;
              }
            }
            S.s_arg[s] = arg;
            atomicAdd(&cnt[arg], 1);
            if (LOG) atomicMin(&S.leader[arg], s);
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
      double t_next = S.red[0];
#pragma unroll
      for (int w = 1; w < NW; ++w) t_next = dmin(t_next, S.red[w]);
      const double dt = __dsub_rn(t_next, now);
      int first_bneck = -1;
      if (LOG && tid == 0 && nA > 0) {
        long long bk = S.red_key[0];
        first_bneck = S.red_id[0];
        for (int w = 1; w < NW; ++w)
          if (S.red_key[w] < bk || (S.red_key[w] == bk && S.red_id[w] < first_bneck)) {
            bk = S.red_key[w];
            first_bneck = S.red_id[w];
          }
      }
      // ======== advance / retire / release (a8).  Also undoes the solve's debits so that link state is back at
      // (cap, n of the surviving flows) for the next event -- exact, because the arithmetic is integer.
      for (int s = tid; s < hi; s += NT) {
        const int f = S.s_flow[s];
        if (f < 0) continue;
        const long long rq = S.s_rq[s];
        const int bn = S.s_bn[s];
        const double rate = rate_of(rq);
        const double rem = S.s_rem[s];
        const double tc = __dadd_rn(now, __ddiv_rn(rem, rate));
        const bool done = tc == t_next;  // bit-equal absolute time (S4.4)
        S.cnt0[bn] = 0;
        S.cnt1[bn] = 0;
        if (LOG) S.leader[bn] = INT_MAX;
        S.s_bn[s] = -1;
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {
          const int l = S.s_path[s * kMaxHops + h];
          if (l < 0) break;
          atomicAdd((unsigned long long *)&S.cap_rem[l], (unsigned long long)rq);
          if (!done) atomicAdd(&S.n[l], 1);
          S.dirty[l] = 1;
        }
        if (done) {
          t_done[f] = t_next;
          bneck_out[f] = bn;
          S.s_flow[s] = -1;
          S.free_stack[atomicAdd(&S.ctl[C_NFREE], 1)] = s;
          atomicSub(&S.ctl[C_NACTIVE], 1);
          atomicAdd(&S.ctl[C_DONE], 1);
          if (LOG) atomicAdd(&S.ctl[C_EV_NCOMP], 1);
          // release successors: pred_cnt--, at 0 -> PENDING with t_act = max(start, now) + Lat (S4.5)
          const uint32_t e0 = rec[f].succ_off, e1 = rec[f + 1].succ_off;
          for (uint32_t e = e0; e < e1; ++e) {
            const int g = succ[e];
            if (atomicSub(&pred_cnt[g], 1) == 1) {
              const FlowRec r = rec[g];
              const double ta = __dadd_rn(r.start > t_next ? r.start : t_next, r.lat);
              const int i = atomicAdd(&S.ctl[C_NP0 + cur], 1);
              if (i < pcap) {
                pf_oth[i] = g;  // pf_oth is the live buffer since the swap after P0
                pt_oth[i] = ta;
              } else {
                S.ctl[C_OVERFLOW] = 1;
              }
            }
          }
        } else {
          const double r2 = __dsub_rn(rem, __dmul_rn(rate, dt));  // mul, then sub, then clamp
          S.s_rem[s] = r2 > 0.0 ? r2 : 0.0;
        }
      }
      if (LOG && tid == 0 && log) {
        phs_event e;
        e.t = t_next;
        e.n_completed = 0;  // n_completed / n_rounds are patched after the next barrier (top of the next P0)
        e.n_activated = S.ctl[C_EV_NACT];
        e.n_rounds = 0;
        e.first_bneck = first_bneck;
        log[n_events] = e;
      }
      if (LOG && tid == 0) S.ctl[C_EV_NACT] = 0;  // next incremented in the next P0, after the barrier below
      now = t_next;
      sum_active += nA;
      sum_rounds += round;
      ++n_events;
      __syncthreads();
    }
    if (tid == 0) {
      if (status == PHS_OK && S.ctl[C_DONE] < F) status = PHS_ECYCLE;  // WAITING flows left over
      InstResult r;
      r.status = status;
      r.path = 0;
      r.n_events = n_events;
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
template <int NT>
static cudaError_t launch_cta_nt(const DevTables &t, const int32_t *order, int n, int *ticket, int acap, int pcap,
                                 int grid, size_t smem, bool log, cudaStream_t stream) {
  cudaError_t e;
  if (log) {
    e = cudaFuncSetAttribute(phs_cta_kernel<NT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    phs_cta_kernel<NT, true><<<grid, NT, smem, stream>>>(t, order, n, ticket, acap, pcap);
  } else {
    e = cudaFuncSetAttribute(phs_cta_kernel<NT, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    phs_cta_kernel<NT, false><<<grid, NT, smem, stream>>>(t, order, n, ticket, acap, pcap);
  }
  return cudaGetLastError();
}

cudaError_t launch_cta_path(const DevTables &t, const int32_t *order, int n, int *ticket, int threads, int acap,
                            int pcap, int grid, size_t smem, bool log, cudaStream_t stream) {
  switch (threads) {
    case 64:
      return launch_cta_nt<64>(t, order, n, ticket, acap, pcap, grid, smem, log, stream);
    case 128:
      return launch_cta_nt<128>(t, order, n, ticket, acap, pcap, grid, smem, log, stream);
    case 256:
      return launch_cta_nt<256>(t, order, n, ticket, acap, pcap, grid, smem, log, stream);
    case 512:
      return launch_cta_nt<512>(t, order, n, ticket, acap, pcap, grid, smem, log, stream);
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
