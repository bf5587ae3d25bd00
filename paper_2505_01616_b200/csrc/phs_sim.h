// phs_sim.h -- the handle behind the C-ABI (struct phs_sim) and the small host helpers shared by phs_api.cu
// (submission calls, result getters) and phs_schedule.cu (table construction, batch scheduler, phs_run).
#pragma once
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstdlib>
#include <deque>
#include <limits>
#include <memory>
#include <string>
#include <thread>
#include <mutex>
#include <exception>
#include <new>
#include <stdexcept>
#include <vector>

#include "phs_device.h"

// records the thread-local error message (phs_last_error) and returns `code`
phs_status phs_fail(phs_status code, const std::string &msg);
struct phs_sim;
// drops the device tables, parked states and results: the next run builds everything again and starts at t = 0
void phs_unfinalize(phs_sim *sim);

#define PHS_CUDA(call)                                                                                       \
  do {                                                                                                       \
    cudaError_t e_ = (call);                                                                                 \
    if (e_ != cudaSuccess) return phs_fail(PHS_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
  } while (0)

// Every extern "C" entry point that returns a status runs between these two: no exception crosses the C-ABI
// (include/phs.h "never throw").  Host allocations (std::vector growth in the submission calls and phs_finalize) are
// the realistic source: they become PHS_ENOMEM.
#define PHS_API_BEGIN try {
#define PHS_API_END                                                       \
  }                                                                       \
  catch (const std::bad_alloc &) {                                        \
    return phs_fail(PHS_ENOMEM, "out of host memory");                    \
  }                                                                       \
  catch (const std::exception &e_) {                                      \
    return phs_fail(PHS_EINVAL, std::string("unexpected exception: ") + e_.what()); \
  }                                                                       \
  catch (...) {                                                           \
    return phs_fail(PHS_EINVAL, "unexpected exception");                  \
  }

namespace phs {

// makes `dev` the current CUDA device for a scope (multi-device handles)
struct DeviceGuard {
  int old = -1;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&old) != cudaSuccess) old = -1;
    cudaSetDevice(dev);
  }
  ~DeviceGuard() {
    if (old >= 0) cudaSetDevice(old);
  }
};

// fn(i) for every i in [0, n) on up to `max_threads` (<= 16) host threads; the iterations must be independent
template <typename F>
void parallel_for(int n, F fn, int max_threads = 16) {
  const int nt = std::min(std::min(n, max_threads), (int)std::min(16u, std::max(1u, std::thread::hardware_concurrency())));
  if (nt <= 1) {
    for (int i = 0; i < n; ++i) fn(i);
    return;
  }
  std::atomic<int> next{0};
  std::exception_ptr err;  // an exception in a worker (std::bad_alloc) is rethrown in the caller, not std::terminate
  std::mutex err_mu;
  std::vector<std::thread> pool;
  for (int t = 0; t < nt; ++t)
    pool.emplace_back([&] {
      try {
        for (int i = next.fetch_add(1); i < n; i = next.fetch_add(1)) fn(i);
      } catch (...) {
        std::lock_guard<std::mutex> g(err_mu);
        if (!err) err = std::current_exception();
        next.store(n);
      }
    });
  for (std::thread &th : pool) th.join();
  if (err) std::rethrow_exception(err);
}

template <typename T>
struct DevBuf {
  T *p = nullptr;
  size_t n = 0;
  bool owned = true;  // false: a view into another allocation (phs_sim::d_arena)
  ~DevBuf() { release(); }
  void release() {
    if (p && owned) cudaFree(p);
    p = nullptr;
    n = 0;
    owned = true;
  }
  void view(T *ptr, size_t count) {
    release();
    p = ptr;
    n = count;
    owned = false;
  }
  cudaError_t alloc(size_t count) {
    release();
    n = count;
    return cudaMalloc((void **)&p, std::max<size_t>(count, 1) * sizeof(T));
  }
  cudaError_t upload(const T *h, size_t count, cudaStream_t st) {
    cudaError_t e = alloc(count);
    if (e != cudaSuccess || count == 0) return e;
    return cudaMemcpyAsync(p, h, count * sizeof(T), cudaMemcpyHostToDevice, st);
  }
  cudaError_t upload(const std::vector<T> &h, cudaStream_t st) { return upload(h.data(), h.size(), st); }
};

// Process-wide page-locked staging area for the tables phs_finalize builds (the per-flow tables are written into
// it by the host threads and copied to HBM at full PCIe / C2C rate).  It grows to the largest request and is
// reused by later handles, so only the first phs_finalize pays for pinning; `mu` is held from the build to the
// end of the copy.  If pinning fails the area is ordinary pageable memory (the copy is slower, nothing else changes).
struct StagingArea {
  std::mutex mu;
  unsigned char *p = nullptr;
  size_t cap = 0;
  bool pinned = false;
  unsigned char *get(size_t bytes) {  // call with `mu` held; nullptr if out of memory
    if (bytes <= cap) return p;
    drop();
    const size_t want = bytes + bytes / 8 + (1u << 20);
    if (cudaHostAlloc((void **)&p, want, cudaHostAllocDefault) == cudaSuccess) {
      pinned = true;
    } else {
      (void)cudaGetLastError();
      p = (unsigned char *)std::malloc(want);
      pinned = false;
    }
    cap = p ? want : 0;
    return p;
  }
  void drop() {
    if (p) {
      if (pinned) cudaFreeHost(p); else std::free(p);
    }
    p = nullptr;
    cap = 0;
  }
};
StagingArea &staging_area();

}  // namespace phs

struct phs_sim {
  phs_topology_desc desc;
  uint64_t seed;
  int32_t batch;
  std::shared_ptr<phs::Fabric> fab;  // immutable after construction: shared with the shards of a multi-device handle
  std::vector<phs::Instance> inst;
  bool want_log = false, finalized = false, ran = false;
  int32_t policy_path = 0, policy_slots = 0;

  // ---- NEXT-4, multi-GPU (phs_set_devices): instances are independent, so a handle bound to several devices is cut
  // into contiguous blocks of instances, one child handle ("shard") per device, built at phs_finalize; runs go to
  // all shards at once (one host thread each), result getters to the shard that holds the instance.
  std::vector<int> devices;
  std::vector<std::unique_ptr<phs_sim>> shards;
  std::vector<int32_t> shard_first;  // [n_shards + 1] first instance of every shard

  // ---- host mirrors built by finalize
  std::vector<int64_t> flow_base;  // [B+1]
  std::vector<int64_t> coll_base;  // [B+1]
  struct Unit {  // what one CTA / cluster simulates (see phs::InstDesc)
    int32_t inst, n_flows, n_links, n_comps;
    int64_t bound;    // upper estimate of the flows PENDING or ACTIVE at once (see phs_finalize)
    int64_t bound_cta;  // the same for the CTA kernel, which reuses a vacated slot within the phase (rings: 1.5 N)
    int64_t bound_whole;  // the part of `bound` from raw flows and all-to-alls (may be in flight all at once)
    int64_t comp_base;    // first entry of the unit in the per-component host arrays (comp_flows, comp_links, h_cown)
    int64_t link_base;    // first entry of the unit in the per-link host arrays (h_lcomp, h_lloc)
    double density;       // estimated flow events per lookahead window (see phs_finalize); decides the window path
    int32_t win_gang;     // CTAs of the unit's gang on the window path, 0 = the unit does not run there
    int32_t win_links, win_comps, win_slots;  // per CTA of the gang: links, components, flow slots (largest member)
  };
  std::vector<Unit> units;
  std::vector<int32_t> unit_first;  // [B+1] units of instance i are unit_first[i] .. unit_first[i+1]-1
  bool decompose = true;
  bool windows = true;  // lookahead-window schedule (phs_set_windows); off: one global event per loop iteration
  double t_stop = 0.0;  // stop time of the current / last run (phs_run_until), +inf for phs_run
  // parked state of the CTA-path units of a run that stopped at parked_until (phs_run_until resumes from it)
  phs::DevBuf<unsigned char> d_park;
  phs::DevBuf<int32_t> d_order2;
  size_t park_stride = 0;
  bool have_park = false;
  int resumed_units = 0;
  // cluster path: parking areas (one launch configuration at a time)
  phs::DevBuf<unsigned char> d_cpark;
  phs::DevBuf<int32_t> d_cpark_index;
  std::vector<int32_t> cpark_index;
  size_t cpark_unit_bytes = 0;
  int cpark_cs = 0, cpark_L = 0;
  int64_t cpark_Sc = 0;
  double parked_until = 0.0;
  // NEXT-1, time rollback: parked states of earlier stop times (phs_set_snapshots), newest last.  A snapshot is
  // everything a resume needs: the parking areas of both kernel paths, the outstanding-predecessor counters, the
  // per-unit result blocks and the length of the history at that time.
  struct Snapshot {
    double t = 0.0;
    phs::DevBuf<unsigned char> park, cpark;
    phs::DevBuf<int32_t> pred_cnt;
    std::vector<phs::InstResult> res;
    unsigned long long hist_n = 0;
    size_t cpark_unit_bytes = 0, n_order = 0, n_cluster = 0;
    int cpark_cs = 0, cpark_L = 0;
    int64_t cpark_Sc = 0;
  };
  std::deque<std::unique_ptr<Snapshot>> snaps;
  int max_snaps = 0;
  double dirty_from = std::numeric_limits<double>::infinity();  // the simulated past is void from this time on
  double resumed_from = 0.0;                                    // time of the state the last run continued from
  std::vector<uint32_t> h_pos;  // output position of a flow -> its position in the per-flow device tables (lazy)
  std::vector<phs::InstDesc> h_desc;  // per unit
  std::vector<phs::InstResult> h_res; // per unit
  std::vector<int32_t> order;  // CTA-path instances, largest first
  std::vector<int32_t> cluster_list;  // instances that go (or fell back) to the cluster path
  // grid path: units that fit no cluster (or all of them under phs_set_scheduler path 4), and its scratch
  std::vector<int32_t> grid_list;
  phs::DevBuf<unsigned char> d_gscratch;
  phs::DevBuf<int32_t> d_glist;
  int grid_ctas = 0;
  // window path: its units, and the ownership tables of their gangs (identity for everybody else)
  std::vector<int32_t> win_list;
  std::vector<int32_t> comp_flows, comp_links, h_lcomp;  // per component: flows, links; per link: its component
  std::vector<uint32_t> h_lloc, h_cown;
  phs::DevBuf<uint32_t> d_lloc, d_cown, d_fcw;
  phs::DevBuf<unsigned long long> d_trel;
  phs::DevBuf<int32_t> d_wlist;
  phs::DevBuf<int> d_wticket;
  int64_t win_scale = 1;  // slot estimate of the window path in quarters of the static bound (doubled after an
                          // overflow): initial flows take their slots only when they are due, so a quarter is typical
  int win_gang_used = 0;
  int64_t total_flows = 0, total_colls = 0;

  // ---- device tables
  phs::DevBuf<unsigned char> d_arena;  // one allocation for every table phs_finalize places (the buffers below are views)
  phs::DevBuf<unsigned char> d_flowtab;  // the per-flow tables (rec, pc0, fmap): allocated before the build, filled group by group
  phs::DevBuf<phs::InstDesc> d_desc;
  phs::DevBuf<phs::FlowRec> d_rec;
  phs::DevBuf<int32_t> d_succ, d_pc0, d_pred_cnt, d_bneck, d_order, d_coll_n, d_linkid;
  phs::DevBuf<uint32_t> d_fmap;
  // throughput history (optional)
  int64_t hist_cap = 0;
  phs::DevBuf<phs::HistRec> d_hist;
  phs::DevBuf<unsigned long long> d_hist_n;
  std::vector<phs::HistRec> h_hist;  // records of the last run, sorted by (flow, event), duplicates of re-runs removed
  phs::DevBuf<int32_t> d_init_f;
  phs::DevBuf<uint8_t> d_pc8;
  phs::DevBuf<int64_t> d_capq, d_coll_first;
  phs::DevBuf<double> d_tdone, d_coll_t, d_init_t;
  phs::DevBuf<phs::InstResult> d_res;
  phs::DevBuf<phs_event> d_log;
  phs::DevBuf<int> d_ticket;
  phs::DevBuf<unsigned char> d_lean;  // CTA path, lean layout: per-CTA global scratch of the working link arrays
  // cluster-path scratch: one region per concurrently running cluster
  phs::DevBuf<uint8_t> g_scratch;
  phs::DevBuf<int32_t> d_clist, d_lcomp;
  phs::DevBuf<int> d_cticket;
  int64_t scratch_Sc = 0, cluster_scale = 1;
  int scratch_regions = 0, scratch_cs = 0, clusters_resident = 0;

  // launch configuration of the CTA path
  phs::CtaLaunch cta{};
  int sm_count = 0;
  size_t smem_optin = 0;
  cudaStream_t last_stream = nullptr;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  int64_t n_launches = 0, h2d_bytes = 0;
  float main_kernel_ms = 0.f;
  ~phs_sim() {
    if (ev0) cudaEventDestroy(ev0);
    if (ev1) cudaEventDestroy(ev1);
  }
};
