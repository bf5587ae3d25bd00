// phs_grid.cu -- grid path of the hot path: the WHOLE GRID simulates one unit (BASELINE.json north_star: "the whole
// grid to each large instance").  For units whose concurrently PENDING + ACTIVE flows do not fit
// the shared memory of a 16-CTA cluster (e.g. a 304-GPU all-to-all: 92,112 concurrent flows).  Same algorithm and
// arithmetic as the other paths (stamp-voting local minima, exact integer shares, lazy settle), but every flow has
// its own state record in global memory (no slot recycling), link state lives in L2-resident global arrays, and the
// phases are separated by cooperative-groups grid barriers: one after phase X, two per filling round.
//
//   X   flows whose time has come complete (results, link counts, DAG release) or activate         | grid barrier
//   V   every flow to re-solve refreshes the shares of its links where they are stale (all flows on
//       a link store the same value), votes for its arg-min link and stamps the others "beaten"    | grid barrier
//   F   flows whose arg-min link is unbeaten freeze, settle and debit their paths (native 64-bit
//       global atomics); every live flow folds its time into the next-event minimum                | grid barrier
//   V / F repeat on the debited shares while flows are left.
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include <climits>
#include <cstdlib>

#include "phs_device.h"
#include "phs_devutil.cuh"

namespace cg = cooperative_groups;

namespace phs {

namespace {

constexpr int NT = kGridThreads;
enum { G_NACT = 0, G_NPEND, G_NDONE, G_LEFT0, G_LEFT1, G_LEFT2, G_ADD0, G_ADD1, G_NCTL };
constexpr int kWaiting = -4, kDone = -3, kPending = -2, kUnfrozen = -1;

__device__ __forceinline__ double block_min(double v, double *red) {
  const unsigned long long b = (unsigned long long)__double_as_longlong(v);
  unsigned hi = (unsigned)(b >> 32), lo = (unsigned)b;
  const unsigned mhi = __reduce_min_sync(0xffffffffu, hi);
  const unsigned mlo = __reduce_min_sync(0xffffffffu, hi == mhi ? lo : 0xffffffffu);
  const double wm = __longlong_as_double((long long)(((unsigned long long)mhi << 32) | mlo));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = wm;
  __syncthreads();
  double m = red[0];
  for (int w = 1; w < NT / 32; ++w) m = dmin(m, red[w]);
  __syncthreads();
  return m;
}

}  // namespace

size_t grid_scratch_bytes(int64_t n_flows, int n_links) {
  const size_t per_flow = 4 * 8 + 2 * 4, per_link = 5 * 8 + 6 * 4;
  return ((size_t)n_flows * per_flow + 255) / 256 * 256 + ((size_t)n_links * per_link + 255) / 256 * 256 + 1024;
}

// HIST: record the throughput history.  The event log is not written on this path.
// INC: incremental re-solve (the same rule as in phs_cluster.cu): an event leaves alone every flow
// whose rate is below the smallest rate it removes from the component and below the smallest floor(cap / n) over the
// links of the flows it adds.  l_caprem then persists from solve to solve (capacity left after ALL frozen flows), a
// completing flow credits its rate back in phase X, the flows at or above the limit credit theirs in a pass of their
// own and are solved by the rounds >= 2 code.
template <bool HIST, bool INC>
__global__ void __launch_bounds__(kGridThreads, 1)
    phs_grid_kernel(DevTables T, const int32_t *__restrict__ list, int n_list, unsigned char *scratch, int64_t max_flows,
                    int max_links) {
  cg::grid_group grid = cg::this_grid();
  const int tid = threadIdx.x;
  const long long gtid = (long long)blockIdx.x * NT + tid, GT = (long long)gridDim.x * NT;
  __shared__ double red[NT / 32];

  // ---- scratch layout (sized by the host for the largest unit of the list)
  size_t o = 0;
  auto take = [&](size_t bytes) {
    unsigned char *p = scratch + o;
    o += (bytes + 15) / 16 * 16;
    return p;
  };
  double *f_tc = (double *)take((size_t)max_flows * 8);    // PENDING: activation time; ACTIVE: completion time
  double *f_rem = (double *)take((size_t)max_flows * 8);
  double *f_tl = (double *)take((size_t)max_flows * 8);
  long long *f_rq = (long long *)take((size_t)max_flows * 8);
  int *f_st = (int *)take((size_t)max_flows * 4);           // kWaiting, kDone, kPending, kUnfrozen, >= 0 bottleneck link
  int *f_arg = (int *)take((size_t)max_flows * 4);
  long long *l_cap = (long long *)take((size_t)max_links * 8);
  long long *l_share0 = (long long *)take((size_t)max_links * 8);
  long long *l_caprem = (long long *)take((size_t)max_links * 8);
  long long *l_sharew = (long long *)take((size_t)max_links * 8);
  int *l_n0 = (int *)take((size_t)max_links * 4);
  int *l_chg = (int *)take((size_t)max_links * 4);
  int *l_beat = (int *)take((size_t)max_links * 4);
  int *l_nw = (int *)take((size_t)max_links * 4);
  int *l_deb = (int *)take((size_t)max_links * 4);
  int *c_solve = (int *)take((size_t)max_links * 4);       // per component (dense ids < links)
  unsigned long long *c_rmin = (unsigned long long *)take((size_t)max_links * 8);  // INC: smallest removed rate
  unsigned long long *gmin = (unsigned long long *)take(4 * 8);
  int *ctl = (int *)take(G_NCTL * 4);

  for (int qi = 0; qi < n_list; ++qi) {
    const int inst = list[qi];
    const InstDesc D = T.inst[inst];
    const FlowRec *__restrict__ rec = T.rec + D.flow_base;
    const int32_t *__restrict__ succ = T.succ + D.succ_base;
    const int32_t *__restrict__ pc0 = T.pred_cnt0 + D.flow_base;
    int32_t *pred_cnt = T.pred_cnt + D.flow_base;
    const uint32_t *__restrict__ fmap = T.fmap + D.flow_base;
    const int64_t *__restrict__ capq = T.capq + D.link_base;
    const int32_t *__restrict__ linkid = T.linkid + D.link_base;
    const int F = D.n_flows, Li = D.n_links;

    // ---- init
    for (long long l = gtid; l < Li; l += GT) {
      l_cap[l] = capq[l];
      l_n0[l] = 0;
      l_chg[l] = 0;
      l_beat[l] = 0;
      l_deb[l] = 0;
      c_solve[l] = 0;
      if (INC) {
        l_caprem[l] = capq[l];
        l_nw[l] = 0;
        c_rmin[l] = ~0ull;
      }
    }
    if (gtid < G_NCTL) ctl[gtid] = 0;
    if (gtid < 3) gmin[gtid] = 0xffffffffffffffffull;
    grid.sync();
    {  // S4: flows without predecessors are PENDING from t = 0 with t_act = start + Lat
      int npend = 0;
      for (long long f = gtid; f < F; f += GT) {
        const int pc = pc0[f];
        pred_cnt[f] = pc;
        f_rq[f] = -1;
        if (pc == 0) {
          const FlowRec r = rec[f];
          f_rem[f] = r.bytes;
          f_tc[f] = __dadd_rn(r.start, r.lat);
          f_st[f] = kPending;
          ++npend;
        } else {
          f_tc[f] = kInf;
          f_st[f] = kWaiting;
        }
      }
      if (npend) atomicAdd(&ctl[G_NPEND], npend);
    }
    __threadfence();
    grid.sync();

    double now = 0.0, t_next = 0.0;
    int ev = -1, solve = 0, g = 0;
    long long sum_active = 0, sum_rounds = 0;
    int max_active = 0, max_pending = 0, status = PHS_OK;

    auto activate = [&](int f, const FlowRec &r) {  // -> ACTIVE: the flow now counts on its links (a4)
#pragma unroll
      for (int h = 0; h < kMaxHops; ++h) {
        const int l = r.path[h];
        if (l < 0) continue;
        atomicAdd(&l_n0[l], 1);
        l_chg[l] = solve;
      }
      c_solve[r.comp] = solve;
      if (INC) ctl[G_ADD0 + (solve & 1)] = 1;  // a flow was added: its links bound what stands (pass A below)
      f_rq[f] = -1;
      f_tc[f] = kInf;
      f_st[f] = kUnfrozen;
    };

    for (;;) {
      if (t_next > T.t_stop) {
        status = kPaused;
        break;
      }
      // ======== phase X (a8 + a4)
      ++solve;
      if (INC && gtid == 0) ctl[G_ADD0 + ((solve + 1) & 1)] = 0;  // last read after the X barrier of the event before
      {
        int d_act = 0, d_pend = 0, d_done = 0;
        for (long long ff = gtid; ff < F; ff += GT) {
          const int f = (int)ff;
          const int st = __ldcg(&f_st[f]);
          if (st == kWaiting || st == kDone) continue;
          if (!(__ldcg(&f_tc[f]) <= t_next)) continue;
          const FlowRec r = rec[f];
          if (st == kPending) {
            activate(f, r);
            ++d_act;
            --d_pend;
            continue;
          }
          // the flow completes at t_next (bit-equal absolute time, S4.4)
          const uint32_t out = fmap[f];
          T.t_done[out] = t_next;
          T.bneck[out] = linkid[st];
          const long long rq_done = INC ? f_rq[f] : 0;
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {
            const int l = r.path[h];
            if (l < 0) continue;
            atomicSub(&l_n0[l], 1);
            l_chg[l] = solve;
            if (INC) atomicAdd((unsigned long long *)&l_caprem[l], (unsigned long long)rq_done);  // its rate goes back
          }
          c_solve[r.comp] = solve;
          if (INC) atomicMin(&c_rmin[r.comp], (unsigned long long)rq_done);
          f_tc[f] = kInf;
          f_st[f] = kDone;
          --d_act;
          ++d_done;
          for (int e = 0; e < r.succ_cnt; ++e) {  // S4.5: release
            const int gs = r.succ_cnt <= 2 ? r.succ_in[e] : succ[r.succ_in[0] + e];
            if (atomicSub(&pred_cnt[gs], 1) != 1) continue;
            const FlowRec rs = rec[gs];
            const double ta = __dadd_rn(rs.start > t_next ? rs.start : t_next, rs.lat);
            f_rem[gs] = rs.bytes;
            if (ta <= t_next) {  // zero path latency: due at this very timestamp
              activate(gs, rs);
              ++d_act;
            } else {
              f_tc[gs] = ta;
              __threadfence();
              f_st[gs] = kPending;
              ++d_pend;
            }
          }
        }
        if (d_act) atomicAdd(&ctl[G_NACT], d_act);
        if (d_pend) atomicAdd(&ctl[G_NPEND], d_pend);
        if (d_done) atomicAdd(&ctl[G_NDONE], d_done);
      }
      __threadfence();
      grid.sync();
      now = t_next;
      ++ev;
      const int nA = __ldcg(&ctl[G_NACT]), nPend = __ldcg(&ctl[G_NPEND]);
      if (nA == 0 && nPend == 0) break;  // S4.3
      max_active = max(max_active, nA);
      max_pending = max(max_pending, nPend);

      // ======== rates (a5-a7)
      auto freeze = [&](int f, int arg, long long rq) {  // a7; R-LZ: only a changed rate touches the flow's state
        f_st[f] = arg;
        const long long old = f_rq[f];
        if (rq != old) {
          double rem = f_rem[f];
          if (old >= 0) {
            rem = __dsub_rn(rem, __dmul_rn(rate_of(old), __dsub_rn(now, f_tl[f])));
            rem = rem > 0.0 ? rem : 0.0;
            f_rem[f] = rem;
          }
          f_tl[f] = now;
          f_rq[f] = rq;
          if (HIST) append_history(T.hist, T.hist_n, T.hist_cap, now, rq, fmap[f], (uint32_t)ev);
          f_tc[f] = __dadd_rn(now, __ddiv_rn(rem, rate_of(rq)));
        }
      };
      int rounds = 0;
      if (INC && __ldcg(&ctl[G_ADD0 + (solve & 1)])) {
        // ---- A: flows were ADDED.  A link that carries an added flow has a share of at least floor(cap / n) -- n its
        // flow count now -- all through the new solve, so the old solve's iterations below the smallest such share are
        // picked again in the same order: every flow slower than that stands.
        for (long long ff = gtid; ff < F; ff += GT) {
          const int f = (int)ff;
          if (__ldcg(&f_st[f]) != kUnfrozen || f_rq[f] >= 0) continue;  // ACTIVE and never solved = added
          const FlowRec r = rec[f];
          long long m = LLONG_MAX;
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {
            const int l = r.path[h];
            if (l < 0) continue;
            const long long sh = fair_share(l_cap[l], __ldcg(&l_n0[l]));
            m = sh < m ? sh : m;
          }
          atomicMin(&c_rmin[r.comp], (unsigned long long)m);
        }
        __threadfence();
        grid.sync();
      }
      if (INC) {  // ---- C: the flows to re-solve give their rates back and count as unfrozen again
        ++g;
        if (gtid == 0) {  // the credit pass takes part in the rotation of the flag / minimum words like a round
          ctl[G_LEFT0 + (g + 1) % 3] = 0;
          gmin[(g + 1) % 3] = 0xffffffffffffffffull;
        }
        for (long long ff = gtid; ff < F; ff += GT) {
          const int f = (int)ff;
          const int st = __ldcg(&f_st[f]);
          if (st == kWaiting || st == kDone || st == kPending) continue;
          const FlowRec r = rec[f];
          if (__ldcg(&c_solve[r.comp]) != solve) continue;  // component untouched by this event: rates stand
          const long long rq = f_rq[f];
          if (rq >= 0 && (unsigned long long)rq < __ldcg(&c_rmin[r.comp])) continue;  // below the limit: stands
          f_st[f] = kUnfrozen;
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {
            const int l = r.path[h];
            if (l < 0) continue;
            if (rq > 0) atomicAdd((unsigned long long *)&l_caprem[l], (unsigned long long)rq);
            atomicAdd(&l_nw[l], 1);
            l_deb[l] = g;  // "debited" in this pass: the next vote computes the link's share from (caprem, nw)
          }
        }
        __threadfence();
        grid.sync();
        for (long long l = gtid; l < Li; l += GT)  // every thread has read the limits: ready for the next event
          if (c_solve[l] == solve) c_rmin[l] = ~0ull;
        rounds = 1;  // the rounds below run as rounds >= 2: shares from the working state, every freeze debits
      }
      for (;;) {
        ++g;
        ++rounds;
        // the flows-left flag and the next-event minimum rotate over three words: round g uses word g mod 3 and
        // clears word (g + 1) mod 3, last read two grid barriers ago
        const int par = g % 3;
        if (gtid == 0) {
          ctl[G_LEFT0 + (g + 1) % 3] = 0;
          gmin[(g + 1) % 3] = 0xffffffffffffffffull;
        }
        // ---- V: shares, arg-min, beat stamps
        for (long long ff = gtid; ff < F; ff += GT) {
          const int f = (int)ff;
          const int st = __ldcg(&f_st[f]);
          if (st == kWaiting || st == kDone || st == kPending) continue;
          const FlowRec r = rec[f];
          if (rounds == 1) {
            if (__ldcg(&c_solve[r.comp]) != solve) continue;  // component untouched by this event: rates stand
          } else if (st != kUnfrozen) {
            continue;
          }
          long long best = LLONG_MAX;
          int arg = -1;
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h) {
            const int l = r.path[h];
            if (l < 0) continue;
            long long sh;
            if (rounds == 1) {
              if (__ldcg(&l_chg[l]) == solve) {  // flow count changed in this event: every flow on l stores the same share
                sh = fair_share(l_cap[l], __ldcg(&l_n0[l]));
                l_share0[l] = sh;
              } else {
                sh = __ldcg(&l_share0[l]);
              }
              l_caprem[l] = l_cap[l];  // working state of the solve's links (idempotent stores; debited from F on)
              l_nw[l] = __ldcg(&l_n0[l]);
              l_sharew[l] = sh;
            } else if (__ldcg(&l_deb[l]) == g - 1) {  // debited in the previous round
              sh = fair_share(__ldcg(&l_caprem[l]), __ldcg(&l_nw[l]));
              l_sharew[l] = sh;
            } else {
              sh = __ldcg(&l_sharew[l]);
            }
            if (sh < best || (sh == best && l < arg)) {
              best = sh;
              arg = l;
            }
          }
#pragma unroll
          for (int h = 0; h < kMaxHops; ++h)
            if (r.path[h] >= 0 && r.path[h] != arg) l_beat[r.path[h]] = g;
          f_arg[f] = arg;
          if (rounds == 1) f_st[f] = kUnfrozen;
        }
        __threadfence();
        grid.sync();
        // ---- F: freeze, settle, debit; fold the times of all live flows
        double mymin = kInf;
        int left = 0;
        for (long long ff = gtid; ff < F; ff += GT) {
          const int f = (int)ff;
          const int st = __ldcg(&f_st[f]);
          if (st == kWaiting || st == kDone) continue;
          if (st == kUnfrozen) {
            const int arg = f_arg[f];
            if (__ldcg(&l_beat[arg]) != g) {
              const long long rq = rounds == 1 ? __ldcg(&l_share0[arg]) : __ldcg(&l_sharew[arg]);
              freeze(f, arg, rq);
              const FlowRec r = rec[f];
#pragma unroll
              for (int h = 0; h < kMaxHops; ++h) {
                const int l = r.path[h];
                if (l < 0) continue;
                if (INC || __ldcg(&l_n0[l]) > 1) {  // INC: caprem persists, so every freeze is booked
                  atomicAdd((unsigned long long *)&l_caprem[l], (unsigned long long)(-rq));
                  atomicSub(&l_nw[l], 1);
                  l_deb[l] = g;
                }
              }
            } else {
              left = 1;
            }
          }
          mymin = dmin(mymin, f_tc[f]);
        }
        left = __syncthreads_or(left);
        const double bm = block_min(mymin, red);
        if (tid == 0) {
          if (left) atomicOr(&ctl[G_LEFT0 + par], 1);
          atomicMin(&gmin[par], (unsigned long long)__double_as_longlong(bm));
        }
        __threadfence();
        grid.sync();
        if (!__ldcg(&ctl[G_LEFT0 + par])) {
          t_next = __longlong_as_double((long long)__ldcg(&gmin[par]));
          break;
        }
      }
      sum_active += nA;
      sum_rounds += rounds;
    }
    if (gtid == 0) {
      InstResult r;
      r.status = status != PHS_OK ? status : (ctl[G_NDONE] < F ? PHS_ECYCLE : PHS_OK);
      r.path = 3;
      r.n_events = ev;
      r.sum_active = sum_active;
      r.sum_par_rounds = sum_rounds;
      r.max_active = max_active;
      r.max_pending = max_pending;
      r.max_slots = max_active + max_pending;
      r.n_windows = ev;
      T.res[inst] = r;
    }
    grid.sync();
  }
}

cudaError_t grid_max_ctas(int *n_ctas) {
  int dev = 0, sms = 0, per = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, phs_grid_kernel<false, true>, kGridThreads, 0);
  if (e != cudaSuccess) return e;
  *n_ctas = sms * std::max(per, 0);
  return cudaSuccess;
}

cudaError_t launch_grid_path(const DevTables &t, const int32_t *list, int n, unsigned char *scratch, int64_t max_flows,
                             int max_links, int n_ctas, cudaStream_t stream) {
  DevTables tt = t;
  void *args[] = {(void *)&tt, (void *)&list, (void *)&n, (void *)&scratch, (void *)&max_flows, (void *)&max_links};
  static const bool inc = [] {  // PHS_GRID_INC=0: from-scratch solves (tuning / comparison runs)
    const char *ev = getenv("PHS_GRID_INC");
    return !(ev && atoi(ev) == 0);
  }();
  const void *fn = inc ? (t.hist ? (const void *)phs_grid_kernel<true, true> : (const void *)phs_grid_kernel<false, true>)
                       : (t.hist ? (const void *)phs_grid_kernel<true, false> : (const void *)phs_grid_kernel<false, false>);
  return cudaLaunchCooperativeKernel(fn, dim3((unsigned)n_ctas), dim3(kGridThreads), args, 0, stream);
}

// ------------------------------------------------------------------------------------------ phs_run_static
// The grid path without any allocation: the kernel's scratch (unit list, per-flow and per-link state) is this
// file-scope array, kStaticScratchBytes on every device that loads the library, held until the process exits.  Every
// call shares it: calls that overlap on one GPU race.  Nothing has to be cleared between calls -- the kernel's init
// phase writes every word it later reads (per unit: link counts, stamps, control words, every flow's state) and the
// unit list is rewritten by phs_static_list_kernel at the start of every call.
static __device__ __align__(256) unsigned char phs_static_scratch[kStaticScratchBytes];

namespace {

// the unit list of a static run is 0 .. n-1, in the first kStaticListBytes of the array (device code names it directly)
__global__ void phs_static_list_kernel(int n) {
  int32_t *list = reinterpret_cast<int32_t *>(phs_static_scratch);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) list[i] = i;
}

// In host code `phs_static_scratch` is a host-side stand-in, not a device address: the address the kernel gets comes
// from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int kMaxStaticDevices = 64;
cudaError_t static_scratch_address(unsigned char **out) {
  static unsigned char *addr[kMaxStaticDevices] = {};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxStaticDevices) return cudaErrorInvalidDevice;
  unsigned char *p = __atomic_load_n(&addr[dev], __ATOMIC_ACQUIRE);
  if (!p) {
    void *sym = nullptr;
    e = cudaGetSymbolAddress(&sym, phs_static_scratch);
    if (e != cudaSuccess) return e;
    if (!sym) return cudaErrorInvalidSymbol;
    p = static_cast<unsigned char *>(sym);
    __atomic_store_n(&addr[dev], p, __ATOMIC_RELEASE);  // every thread gets the same answer for one device
  }
  *out = p;
  return cudaSuccess;
}

}  // namespace

size_t grid_static_capacity() { return kStaticScratchBytes - kStaticListBytes; }

cudaError_t launch_grid_static(const DevTables &t, int n_units, int64_t max_flows, int max_links, int n_ctas,
                               cudaStream_t stream) {
  if (n_units < 1 || (size_t)n_units * sizeof(int32_t) > kStaticListBytes ||
      grid_scratch_bytes(max_flows, max_links) > grid_static_capacity())
    return cudaErrorInvalidValue;  // the caller (phs_run_static) checks first and says which limit it was
  unsigned char *base = nullptr;
  cudaError_t e = static_scratch_address(&base);
  if (e != cudaSuccess) return e;
  phs_static_list_kernel<<<(n_units + 255) / 256, 256, 0, stream>>>(n_units);
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  return launch_grid_path(t, reinterpret_cast<const int32_t *>(base), n_units, base + kStaticListBytes, max_flows,
                          max_links, n_ctas, stream);
}

}  // namespace phs
