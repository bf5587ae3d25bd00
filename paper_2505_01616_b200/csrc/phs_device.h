// phs_device.h -- kernel-side table of device pointers and the launch entry points of the four kernel paths
// (phs_kernels.cu, phs_cluster.cu, phs_window.cu, phs_grid.cu), called from phs_schedule.cu.
#pragma once
#include <cuda_runtime.h>

#include "phs_internal.h"

namespace phs {

struct HistRec {     // one rate change of one flow (throughput history, PAPER.md L128 / L167)
  double t;          // when
  double rate;       // new rate, byte/s
  uint32_t flow;     // position of the flow in t_done[] / bneck[]
  uint32_t ev;       // index of the unit's event that changed it (orders changes at one and the same time)
};

struct ParkRegs {  // the loop-carried registers of a parked unit (CTA path)
  double now, t_next;
  long long sum_active, sum_rounds;
  int32_t ev, solve, g, max_active, max_pending, first_bneck, valid, n_windows;
};

struct DevTables {
  const InstDesc *inst;      // [U] simulation units
  const FlowRec *rec;        // [F_total] unit-local link / flow ids inside
  const int32_t *succ;       // successor lists longer than two (unit-local flow ids)
  const int32_t *pred_cnt0;  // [F_total] number of predecessors
  const uint8_t *pred_cnt0_u8;  // same, packed 4 bits per flow (per-unit slices 4-byte aligned); unused if a count > 15
  const uint32_t *fmap;      // [F_total] unit-local flow -> index of the flow in t_done[] / bneck[]
  const double *init_t;      // per unit [n_init] activation times start + Lat of the flows without predecessors,
  const int32_t *init_f;     //   ascending (ties by flow id), and the flows themselves (cluster path: these flows
                             //   take a slot only when they activate)
  const int64_t *capq;       // per unit [n_links] link capacity in rate quanta
  const int32_t *lcomp;      // per unit [n_links] static component (representative unit-local link) of every link
  const int32_t *linkid;     // per unit [n_links] unit-local link -> link id of the topology
  int32_t *pred_cnt;         // [F_total] outstanding predecessors (dynamic)
  double *t_done;            // [F_total] O1, in the caller's flow order
  int32_t *bneck;            // [F_total] O3, topology link ids
  InstResult *res;           // [U]
  phs_event *log;            // event log rows, or nullptr
  HistRec *hist;             // throughput history records, or nullptr
  unsigned long long *hist_n;  // records produced (may exceed hist_cap: the excess is dropped and reported)
  long long hist_cap;
  double t_stop;             // phs_run_until: stop before the first event later than this (+inf: run to the end)
  unsigned char *park;       // CTA path: per unit, ParkRegs + a copy of the CTA's dynamic shared memory, written
  size_t park_stride;        //   when a unit stops at t_stop so that a later phs_run_until can resume it; or nullptr
  int32_t resume;            // 1: units with a valid parked state continue from it instead of starting at t = 0
  int32_t n_links;           // largest n_links among the units of this launch (sizes the shared-memory layout)
  // window path: which CTA of the gang owns what (for the gang size the scheduler chose for the unit)
  const uint32_t *lloc;      // per unit [n_links]: owner CTA << 24 | index of the link in the owner's shared memory
  const uint32_t *cown;      // per unit [n_comps]: owner CTA << 24 | index of the component in the owner
  unsigned long long *t_rel; // [F_total] scratch: latest completion time (bit pattern) among a flow's predecessors
  uint32_t *fcw;             // [F_total] scratch: cown of the flow's component
};

// Shared-memory footprint of the CTA kernel for given capacities (pc_flows > 0: predecessor counters of that
// many flows are kept in shared memory as bytes).
size_t cta_smem_bytes(int n_links, int slots, int pc_flows, bool log, int lean = 0);
size_t cta_lean_scratch_bytes(int n_links);  // global scratch per CTA of a lean launch

// One CTA per instance (persistent CTAs pull instance indices from order[0..n) through *ticket).
// Instances that run out of shared-memory slots finish with status kOverflow.
struct CtaLaunch {
  int threads, slots, pc_flows, grid;
  int n_links;  // largest link count among the units of the launch
  size_t smem;
  bool log;
  // Lean shared-memory layout, for batches with many times more units than can be resident (the SMs' issue slots are
  // the limit and every further resident CTA hides latency): bit 0 = the per-link arrays that only a solve with a
  // second filling round touches, and the link ids, live in global memory (lean_scratch: grid * cta_lean_scratch_bytes,
  // L2-resident) and in the unit's tables; bit 1 = so do the capacities.  0 = everything in shared memory.
  int lean;
  unsigned char *lean_scratch;
};
cudaError_t launch_cta_path(const DevTables &t, const int32_t *order, int n, int *ticket, const CtaLaunch &cfg,
                            cudaStream_t stream);

// Cluster path (phs_cluster.cu): one thread-block cluster (1-16 CTAs, hardware cluster barrier) per unit that does not
// fit one SM.  All dynamic state stays on chip: link l is owned by CTA (l mod cluster size) and lives in the owner's
// shared memory, reached by the others through distributed shared memory; every CTA owns private flow slots in its own
// shared memory (only the cold slot fields spill to `base`, a CTA-private global partition, when shared memory is
// short).  Clusters pull unit indices from list[0..n) through *ticket; the cluster with rank k in the grid uses spill
// region k.
struct ClusterScratch {
  unsigned char *base;  // global spill area of the cold slot fields (n_regions * region_bytes), unused if cold_smem
  size_t region_bytes;
  int64_t Sc;           // flow slots per CTA
  int aggregate;        // 1: a CTA pre-sums its debits per link in shared memory (16 bytes per link and CTA)
  int cold_smem;        // 1: the cold slot fields live in shared memory too
  int replicate;        // 1: every CTA keeps a copy of the links' current fair shares (22 bytes per link and CTA)
  int incremental;      // 1 (needs aggregate and replicate, no event log): an event that only removes flows re-solves
                        // just the flows whose rate is at least the smallest removed rate (phs_cluster.cu, INC)
  // phs_run_until: parking areas of units that stopped at t_stop (per unit: ClusterParkRegs, then per CTA a copy
  // of its shared memory, control words and cold slot fields), or nullptr
  unsigned char *park;
  size_t park_unit_stride, park_cta_stride;
  const int32_t *park_index;  // [units] index of the unit's parking area, -1 = none
  int resume;                 // 1: units with a valid parked state continue from it
};
struct ClusterParkRegs {  // the loop-carried registers of a parked unit (cluster path)
  double now, t_next, t_init;
  long long sum_active, sum_rounds;
  int32_t ev, solve, g, ip, n_done, prev_nact, max_active, max_pending, max_slots, first_bneck, valid, pad_;
};
constexpr size_t kClusterParkHeader = 256;  // bytes reserved for ClusterParkRegs at the start of a unit's area
size_t cluster_park_cta_bytes(int n_links, int cluster_size, int64_t Sc, bool aggregate, bool cold_smem, bool log,
                              bool replicate);
constexpr int kClusterThreads = 512;
// dynamic shared memory per CTA / global spill bytes per cluster
size_t cluster_smem_bytes(int n_links, int cluster_size, int64_t Sc, bool aggregate, bool cold_smem, bool log,
                          bool replicate);
size_t cluster_region_bytes(int64_t Sc, int cluster_size);
// how many clusters of this size and shared-memory footprint can be resident at once (0: it cannot launch)
cudaError_t cluster_max_clusters(int cluster_size, size_t smem, int *max_clusters);
cudaError_t launch_cluster_path(const DevTables &t, const int32_t *list, int n, int *ticket, const ClusterScratch &s,
                                int cluster_size, int n_clusters, bool log, cudaStream_t stream);

// Window path (phs_window.cu): one gang (thread-block cluster of `gang` CTAs, kWindowThreads threads each) per unit;
// the unit's static link components are partitioned over the CTAs (lloc / cown in DevTables), every CTA keeps the
// links, components and flow slots it owns in its own shared memory and the gang meets only at the end of a
// lookahead window.  Gangs pull units from list[0..n) through *ticket.
constexpr int kWindowThreads = 256;
struct WindowLaunch {
  int gang;     // CTAs per unit: 1, 2, 4, 8 or 16
  int slots;    // flow slots per CTA
  int n_links;  // links per CTA (largest over the units of the launch and their CTAs)
  int n_comps;  // components per CTA (likewise)
  size_t smem;  // dynamic shared memory per CTA
};
size_t window_smem_bytes(int n_links, int n_comps, int slots);
cudaError_t window_max_clusters(int gang, size_t smem, int *max_clusters);
cudaError_t launch_window_path(const DevTables &t, const int32_t *list, int n, int *ticket, const WindowLaunch &w,
                               int n_clusters, cudaStream_t stream);

// Grid path (phs_grid.cu): the whole grid (cooperative launch, n_ctas CTAs of kGridThreads threads) simulates the
// units of list[0..n) one after the other; per-flow and per-link state in `scratch` (grid_scratch_bytes for the
// largest unit of the list).
constexpr int kGridThreads = 512;
size_t grid_scratch_bytes(int64_t n_flows, int n_links);
cudaError_t grid_max_ctas(int *n_ctas);
cudaError_t launch_grid_path(const DevTables &t, const int32_t *list, int n, unsigned char *scratch, int64_t max_flows,
                             int max_links, int n_ctas, cudaStream_t stream);

// phs_run_static: the same kernel with its scratch (and the unit list 0 .. n_units-1) in a file-scope __device__ array
// of kStaticScratchBytes; allocates nothing.  cudaErrorInvalidValue if the list or the state does not fit.
constexpr size_t kStaticScratchBytes = PHS_STATIC_SCRATCH_BYTES;
constexpr size_t kStaticListBytes = (size_t)PHS_STATIC_MAX_UNITS * sizeof(int32_t);
size_t grid_static_capacity();  // bytes left for per-flow / per-link state (grid_scratch_bytes must not exceed it)
cudaError_t launch_grid_static(const DevTables &t, int n_units, int64_t max_flows, int max_links, int n_ctas,
                               cudaStream_t stream);

// NEXT-1: forgets the results later than t (t_done = NaN, bneck = -1)
cudaError_t launch_forget_after(double *t_done, int32_t *bneck, int64_t n, double t, cudaStream_t stream);

// out[c] = max t_done over the flows of collective c, for all collectives of all instances.
cudaError_t launch_collective_times(const double *t_done, const int64_t *coll_first, const int32_t *coll_nflows,
                                    int64_t n_colls, double *out, cudaStream_t stream);

}  // namespace phs
