// phs_device.h -- kernel-side table of device pointers and the launch entry points (implemented in
// phs_kernels.cu, called from phs_api.cu).
#pragma once
#include <cuda_runtime.h>

#include "phs_internal.h"

namespace phs {

struct DevTables {
  const InstDesc *inst;      // [B]
  const FlowRec *rec;        // [F_total]
  const int32_t *succ;       // successor CSR values (instance-relative flow ids)
  const int32_t *pred_cnt0;  // [F_total] number of predecessors
  const uint8_t *pred_cnt0_u8;  // same as bytes (per-instance slices 4-byte aligned), or nullptr if a count > 255
  const int64_t *capq;       // [B][n_links] link capacity in rate quanta
  int32_t *pred_cnt;         // [F_total] outstanding predecessors (dynamic)
  double *t_done;            // [F_total] O1
  int32_t *bneck;            // [F_total] O3
  InstResult *res;           // [B]
  phs_event *log;            // event log rows, or nullptr
  int32_t n_links;
};

// Shared-memory footprint of the CTA kernel for given capacities (pc_flows > 0: predecessor counters of that
// many flows are kept in shared memory as bytes).
size_t cta_smem_bytes(int n_links, int slots, int pc_flows, bool log);

// One CTA per instance (persistent CTAs pull instance indices from order[0..n) through *ticket).
// Instances that run out of shared-memory slots finish with status kOverflow.
struct CtaLaunch {
  int threads, slots, pc_flows, grid;
  size_t smem;
  bool log;
};
cudaError_t launch_cta_path(const DevTables &t, const int32_t *order, int n, int *ticket, const CtaLaunch &cfg,
                            cudaStream_t stream);

// Cluster path: one thread-block cluster (up to 16 CTAs, hardware cluster barrier) per large instance, all state
// in global memory (L2-resident).  Clusters pull instance indices from list[0..n) through *ticket; the cluster
// with rank k in the grid uses scratch region k.
struct ClusterScratch {
  int64_t *i64;   // per region: cap_rem[L], share[L], a_rq[Fs]
  int32_t *i32;   // per region: n, nsnap, cnt0, cnt1, leader [L each]; a_flow, a_bn, a_arg, free_stack, p_flow0,
                  //             p_flow1 [Fs each]; a_path [kMaxHops * Fs]
  double *f64;    // per region: a_rem, p_tact0, p_tact1, a_tl, a_tc [Fs each]
  uint8_t *u8;    // per region: dirty[L]
  unsigned long long *ctrl;  // per region: 64 words of control state
  int64_t Fs;     // slot capacity of a region (>= flows of the largest instance on this path)
};
__host__ __device__ inline size_t cluster_i64_per_region(int L, int64_t Fs) { return (size_t)(2 * (int64_t)L + Fs); }
__host__ __device__ inline size_t cluster_i32_per_region(int L, int64_t Fs) { return (size_t)(5 * (int64_t)L + (6 + kMaxHops) * Fs); }
__host__ __device__ inline size_t cluster_f64_per_region(int64_t Fs) { return (size_t)(5 * Fs); }
constexpr int kClusterThreads = 1024;
// Largest cluster size (<= want) that can be co-scheduled, and how many such clusters fit on the device at once.
cudaError_t cluster_path_limits(int want, int *cluster_size, int *max_clusters);
cudaError_t launch_cluster_path(const DevTables &t, const int32_t *list, int n, int *ticket, const ClusterScratch &s,
                                int cluster_size, int n_clusters, bool log, cudaStream_t stream);

// out[c] = max t_done over the flows of collective c, for all collectives of all instances.
cudaError_t launch_collective_times(const double *t_done, const int64_t *coll_first, const int32_t *coll_nflows,
                                    int64_t n_colls, double *out, cudaStream_t stream);

}  // namespace phs
