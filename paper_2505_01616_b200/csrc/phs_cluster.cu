// phs_cluster.cu -- cluster path of the hot path: one thread-block cluster (up to 16 CTAs x 1024 threads, hardware
// cluster barrier) simulates one LARGE instance; all state lives in global memory (L2-resident).  Same algorithm
// and the same three phases per filling round as the CTA path (phs_kernels.cu); what changes is the barrier
// (barrier.cluster with release/acquire) and that votes / debits are global (L2) atomics.
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include <climits>

#include "phs_device.h"
#include "phs_devutil.cuh"

namespace cg = cooperative_groups;

namespace phs {

namespace {

// control block of one scratch region, viewed as int[128]; words 64.. hold 64-bit values
enum {
  K_HI = 0, K_NFREE, K_NP0, K_NP1, K_NACTIVE, K_DONE, K_EV_NACT, K_EV_NCOMP, K_EV_ROUNDS, K_LEFT0, K_LEFT1, K_LEFT2,
  K_INST, K_FB_ID0 = 16 /* 16 per-CTA first_bneck ids */, K_NWORDS32 = 32
};
// 64-bit words (index into unsigned long long ctrl[]): [16],[17] = t_next minima by event parity,
// [32..48) = per-CTA first_bneck keys
constexpr int Q_TMIN0 = 16, Q_FB_KEY0 = 32;

__device__ __forceinline__ int ld_ctl(const int *p) { return *(const volatile int *)p; }

}  // namespace

template <bool LOG>
__global__ void __launch_bounds__(kClusterThreads, 1)
    phs_cluster_kernel(DevTables T, const int32_t *__restrict__ list, int n_list, int *ticket, ClusterScratch SC) {
  cg::cluster_group cluster = cg::this_cluster();
  const int CS = (int)cluster.num_blocks();
  const int crank = (int)cluster.block_rank();
  const int region = blockIdx.x / CS;
  constexpr int NT = kClusterThreads;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int ctid = crank * NT + tid;  // thread index within the cluster
  const int CT = CS * NT;             // threads in the cluster
  const int L = T.n_links;
  const int64_t Fs = SC.Fs;

  // ---- carve this cluster's scratch region
  long long *cap_rem = (long long *)SC.i64 + (size_t)region * cluster_i64_per_region(L, Fs);
  long long *share = cap_rem + L;
  long long *a_rq = share + L;
  int *nl = SC.i32 + (size_t)region * cluster_i32_per_region(L, Fs);
  int *nsnap = nl + L, *cnt0 = nsnap + L, *cnt1 = cnt0 + L, *leader = cnt1 + L;
  int *a_flow = leader + L;
  int *a_bn = a_flow + Fs, *a_arg = a_bn + Fs, *free_stack = a_arg + Fs;
  int *p_flow0 = free_stack + Fs, *p_flow1 = p_flow0 + Fs;
  int *a_path = p_flow1 + Fs;
  double *a_rem = SC.f64 + (size_t)region * cluster_f64_per_region(Fs);
  double *p_tact0 = a_rem + Fs, *p_tact1 = p_tact0 + Fs;
  double *a_tl = p_tact1 + Fs, *a_tc = a_tl + Fs;  // R-LZ: time of the last rate change, completion time
  unsigned char *dirty = SC.u8 + (size_t)region * L;
  unsigned long long *ctrl64 = SC.ctrl + (size_t)region * 64;
  int *ctl = (int *)ctrl64;

  __shared__ double red[32];
  __shared__ long long red_key[32];
  __shared__ int red_id[32];

  for (;;) {
    // ---- a9: clusters pull instances from the list
    if (ctid == 0) ctl[K_INST] = atomicAdd(ticket, 1);
    cluster.sync();
    const int qi = ld_ctl(&ctl[K_INST]);
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
    phs_event *log = (LOG && D.log_base >= 0) ? T.log + D.log_base : nullptr;
    const int F = D.n_flows;

    // ---- init (S4): full capacities, nothing active, flows without predecessors PENDING
    for (int l = ctid; l < L; l += CT) {
      cap_rem[l] = capq[l];
      nl[l] = 0;
      cnt0[l] = 0;
      cnt1[l] = 0;
      leader[l] = INT_MAX;
      dirty[l] = 0;
    }
    if (ctid < K_INST) ctl[ctid] = 0;
    if (ctid == 0) {
      ctrl64[Q_TMIN0] = (unsigned long long)__double_as_longlong(kInf);
      ctrl64[Q_TMIN0 + 1] = (unsigned long long)__double_as_longlong(kInf);
    }
    cluster.sync();
    for (int f = ctid; f < F; f += CT) {
      const int pc = pc0[f];
      pred_cnt[f] = pc;
      if (pc == 0) {
        const FlowRec r = rec[f];
        const int i = atomicAdd(&ctl[K_NP0], 1);
        p_flow0[i] = f;
        p_tact0[i] = __dadd_rn(r.start, r.lat);
      }
    }
    cluster.sync();

    double now = 0.0;
    int cur = 0;
    long long n_events = 0, sum_active = 0, sum_rounds = 0;
    int max_active = 0, max_pending = 0;

    for (;;) {
      // ======== P0 (a4): activate PENDING flows with t_act <= now
      const int nP = ld_ctl(&ctl[K_NP0 + cur]);
      int *const pf_cur = cur ? p_flow1 : p_flow0, *const pf_oth = cur ? p_flow0 : p_flow1;
      double *const pt_cur = cur ? p_tact1 : p_tact0, *const pt_oth = cur ? p_tact0 : p_tact1;
      double mymin = kInf;
      for (int i = ctid; i < nP; i += CT) {
        const int f = pf_cur[i];
        const double ta = pt_cur[i];
        if (ta <= now) {
          int slot;
          const int k = atomicSub(&ctl[K_NFREE], 1) - 1;
          if (k >= 0)
            slot = free_stack[k];
          else
            slot = atomicAdd(&ctl[K_HI], 1);
          const FlowRec r = rec[f];
          a_flow[slot] = f;
          a_rem[slot] = r.bytes;
          a_rq[slot] = -1;  // no rate yet
          a_tc[slot] = kInf;
          a_bn[slot] = -1;
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {
            const int l = r.path[h];
            if (l >= 0) {
              atomicAdd(&nl[l], 1);
              dirty[l] = 1;
            }
            a_path[(size_t)slot * kMaxHops + h] = l;
          }
          atomicAdd(&ctl[K_NACTIVE], 1);
          if (LOG) atomicAdd(&ctl[K_EV_NACT], 1);
        } else {
          const int j = atomicAdd(&ctl[K_NP0 + (cur ^ 1)], 1);
          pf_oth[j] = f;
          pt_oth[j] = ta;
          mymin = dmin(mymin, ta);
        }
      }
      cluster.sync();
      if (ctid == 0) {
        ctl[K_NP0 + cur] = 0;
        if (ld_ctl(&ctl[K_NFREE]) < 0) ctl[K_NFREE] = 0;
        if (LOG) {
          if (log && n_events > 0) {
            log[n_events - 1].n_completed = ld_ctl(&ctl[K_EV_NCOMP]);
            log[n_events - 1].n_rounds = ld_ctl(&ctl[K_EV_ROUNDS]);
          }
          ctl[K_EV_NCOMP] = 0;
          ctl[K_EV_ROUNDS] = 0;
        }
      }
      cur ^= 1;
      const int nA = ld_ctl(&ctl[K_NACTIVE]);
      const int nPend = ld_ctl(&ctl[K_NP0 + cur]);
      if (nA == 0 && nPend == 0) break;
      const int hi = ld_ctl(&ctl[K_HI]);
      max_active = max(max_active, nA);
      max_pending = max(max_pending, nPend);
      const int par = (int)(n_events & 1);

      // ======== rates (a5-a7): parallel progressive filling, candidate completion times folded in (a8)
      int round = 0, it = 0;
      bool left = nA > 0;
      for (;;) {
        if (left) {
          int *cnt = (round & 1) ? cnt1 : cnt0;
          int *cnt_prev = (round & 1) ? cnt0 : cnt1;
          // (a) fair share of every link whose (cap_rem, n) changed
          long long bk = LLONG_MAX;
          int bl = INT_MAX;
          for (int l = ctid; l < L; l += CT) {
            const int nn = nl[l];
            if (dirty[l]) {
              dirty[l] = 0;
              nsnap[l] = nn;
              if (nn > 0) share[l] = fair_share(cap_rem[l], nn);
            }
            if (LOG && round == 0 && nn > 0) {
              const long long sh = share[l];
              if (sh < bk) {
                bk = sh;
                bl = l;
              }
            }
          }
          if (LOG && round == 0) {  // first_bneck: per-CTA partial, combined by thread 0 of the cluster later
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
              ctrl64[Q_FB_KEY0 + crank] = (unsigned long long)bk;
              ctl[K_FB_ID0 + crank] = bl;
            }
          }
          cluster.sync();
          // (b) every unfrozen flow votes for the arg-min link of its path
          for (int s = ctid; s < hi; s += CT) {
            if (a_flow[s] < 0 || a_bn[s] >= 0) continue;
            if (round > 0) cnt_prev[a_arg[s]] = 0;
            long long best = LLONG_MAX;
            int arg = -1;
#pragma unroll
            for (int h = 0; h < kMaxHops; ++h) {
              const int l = a_path[(size_t)s * kMaxHops + h];
              if (l < 0) break;
              const long long sh = share[l];
              if (sh < best || (sh == best && l < arg)) {
                best = sh;
                arg = l;
              }
            }
            a_arg[s] = arg;
            atomicAdd(&cnt[arg], 1);
            if (LOG) atomicMin(&leader[arg], s);
          }
          cluster.sync();
          // (c) links that collected the votes of all their unfrozen flows freeze them; debit the paths
          bool mine_left = false;
          for (int s = ctid; s < hi; s += CT) {
            if (a_flow[s] < 0 || a_bn[s] >= 0) continue;
            const int arg = a_arg[s];
            if (cnt[arg] == nsnap[arg]) {
              const long long rq = share[arg];
              const long long old = a_rq[s];
              a_bn[s] = arg;
              if (rq != old) {  // R-LZ: only a changed rate touches the flow: settle, then a new completion time
                double rem = a_rem[s];
                if (old >= 0) {
                  rem = __dsub_rn(rem, __dmul_rn(rate_of(old), __dsub_rn(now, a_tl[s])));
                  rem = rem > 0.0 ? rem : 0.0;
                  a_rem[s] = rem;
                }
                a_tl[s] = now;
                a_rq[s] = rq;
                a_tc[s] = __dadd_rn(now, __ddiv_rn(rem, rate_of(rq)));
              }
#pragma unroll
              for (int h = 0; h < kMaxHops; ++h) {
                const int l = a_path[(size_t)s * kMaxHops + h];
                if (l < 0) break;
                atomicAdd((unsigned long long *)&cap_rem[l], (unsigned long long)(-rq));
                atomicSub(&nl[l], 1);
                dirty[l] = 1;
              }
              mymin = dmin(mymin, a_tc[s]);
              if (LOG && leader[arg] == s) atomicAdd(&ctl[K_EV_ROUNDS], 1);
            } else {
              mine_left = true;
              if (LOG) leader[arg] = INT_MAX;
            }
          }
          left = mine_left;
          ++round;
        }
        // cluster-wide: t_next candidate minimum and "any flow still unfrozen"
        const double wm = warp_min(mymin);
        if (lane == 0) red[warp] = wm;
        const int cta_left = __syncthreads_or(left);
        if (tid == 0) {
          double m = red[0];
          for (int w = 1; w < NT / 32; ++w) m = dmin(m, red[w]);
          atomicMin(&ctrl64[Q_TMIN0 + par], (unsigned long long)__double_as_longlong(m));
          if (cta_left) *(volatile int *)&ctl[K_LEFT0 + it % 3] = 1;
          if (crank == 0) *(volatile int *)&ctl[K_LEFT0 + (it + 2) % 3] = 0;  // last read two barriers ago
        }
        cluster.sync();
        left = ld_ctl(&ctl[K_LEFT0 + it % 3]) != 0;
        ++it;
        if (!left) break;
      }
      // ======== next time (a8)
      const double t_next = __longlong_as_double((long long)*(volatile unsigned long long *)&ctrl64[Q_TMIN0 + par]);
      int first_bneck = -1;
      if (LOG && ctid == 0 && nA > 0) {
        long long bk = LLONG_MAX;
        for (int c = 0; c < CS; ++c) {
          const long long k = (long long)*(volatile unsigned long long *)&ctrl64[Q_FB_KEY0 + c];
          const int id = ld_ctl(&ctl[K_FB_ID0 + c]);
          if (k < bk || (k == bk && id < first_bneck)) {
            bk = k;
            first_bneck = id;
          }
        }
      }
      // ======== advance / retire / release (a8); restores link state exactly (integer arithmetic)
      for (int s = ctid; s < hi; s += CT) {
        const int f = a_flow[s];
        if (f < 0) continue;
        const long long rq = a_rq[s];
        const int bn = a_bn[s];
        const bool done = a_tc[s] == t_next;
        cnt0[bn] = 0;
        cnt1[bn] = 0;
        if (LOG) leader[bn] = INT_MAX;
        a_bn[s] = -1;
#pragma unroll
        for (int h = 0; h < kMaxHops; ++h) {
          const int l = a_path[(size_t)s * kMaxHops + h];
          if (l < 0) break;
          atomicAdd((unsigned long long *)&cap_rem[l], (unsigned long long)rq);
          if (!done) atomicAdd(&nl[l], 1);
          dirty[l] = 1;
        }
        if (done) {
          t_done[f] = t_next;
          bneck_out[f] = bn;
          a_flow[s] = -1;
          free_stack[atomicAdd(&ctl[K_NFREE], 1)] = s;
          atomicSub(&ctl[K_NACTIVE], 1);
          atomicAdd(&ctl[K_DONE], 1);
          if (LOG) atomicAdd(&ctl[K_EV_NCOMP], 1);
          const int nsucc = rec[f].succ_cnt;
          const int s0 = rec[f].succ_in[0], s1 = rec[f].succ_in[1];
          for (int e = 0; e < nsucc; ++e) {
            const int g = nsucc <= 2 ? (e == 0 ? s0 : s1) : succ[s0 + e];
            if (atomicSub(&pred_cnt[g], 1) == 1) {
              const FlowRec r = rec[g];
              const double ta = __dadd_rn(r.start > t_next ? r.start : t_next, r.lat);
              const int i = atomicAdd(&ctl[K_NP0 + cur], 1);
              pf_oth[i] = g;  // pf_oth is the live buffer since the swap after P0
              pt_oth[i] = ta;
            }
          }
        }
      }
      if (ctid == 0) {
        if (LOG && log) {
          phs_event e;
          e.t = t_next;
          e.n_completed = 0;  // patched after the next barrier (top of the next P0)
          e.n_activated = ld_ctl(&ctl[K_EV_NACT]);
          e.n_rounds = 0;
          e.first_bneck = first_bneck;
          log[n_events] = e;
        }
        if (LOG) ctl[K_EV_NACT] = 0;
        ctl[K_LEFT0] = 0;
        ctl[K_LEFT1] = 0;
        ctl[K_LEFT2] = 0;
        ctrl64[Q_TMIN0 + (par ^ 1)] = (unsigned long long)__double_as_longlong(kInf);
      }
      now = t_next;
      sum_active += nA;
      sum_rounds += round;
      ++n_events;
      cluster.sync();
    }
    if (ctid == 0) {
      InstResult r;
      r.status = ld_ctl(&ctl[K_DONE]) < F ? PHS_ECYCLE : PHS_OK;
      r.path = 1;
      r.n_events = n_events;
      r.sum_active = sum_active;
      r.sum_par_rounds = sum_rounds;
      r.max_active = max_active;
      r.max_pending = max_pending;
      T.res[inst] = r;
    }
    cluster.sync();
  }
}

// ------------------------------------------------------------------------------------------------ launch
namespace {
void set_cluster_attr(cudaLaunchConfig_t &cfg, cudaLaunchAttribute *attr, int cluster_size, int n_clusters,
                      cudaStream_t stream) {
  cfg.gridDim = dim3((unsigned)(cluster_size * n_clusters));
  cfg.blockDim = dim3(kClusterThreads);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = stream;
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)cluster_size;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
}

template <bool LOG>
cudaError_t launch_cluster_t(const DevTables &t, const int32_t *list, int n, int *ticket, const ClusterScratch &s,
                             int cluster_size, int n_clusters, cudaStream_t stream) {
  cudaError_t e = cudaFuncSetAttribute(phs_cluster_kernel<LOG>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg{};
  cudaLaunchAttribute attr[1];
  set_cluster_attr(cfg, attr, cluster_size, n_clusters, stream);
  return cudaLaunchKernelEx(&cfg, phs_cluster_kernel<LOG>, t, list, n, ticket, s);
}
}  // namespace

cudaError_t launch_cluster_path(const DevTables &t, const int32_t *list, int n, int *ticket, const ClusterScratch &s,
                                int cluster_size, int n_clusters, bool log, cudaStream_t stream) {
  return log ? launch_cluster_t<true>(t, list, n, ticket, s, cluster_size, n_clusters, stream)
             : launch_cluster_t<false>(t, list, n, ticket, s, cluster_size, n_clusters, stream);
}

cudaError_t cluster_path_limits(int want, int *cluster_size, int *max_clusters) {
  cudaError_t e = cudaFuncSetAttribute(phs_cluster_kernel<false>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(phs_cluster_kernel<true>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (e != cudaSuccess) return e;
  for (int cs = want; cs >= 1; cs >>= 1) {
    cudaLaunchConfig_t cfg{};
    cudaLaunchAttribute attr[1];
    set_cluster_attr(cfg, attr, cs, 1, nullptr);
    int n = 0;
    e = cudaOccupancyMaxActiveClusters(&n, phs_cluster_kernel<true>, &cfg);
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
