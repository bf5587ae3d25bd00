// phs_internal.h -- shared between the host builder (phs_build.cpp), the API (phs_api.cu) and the kernels
// (phs_kernels.cu).  Nothing here is shared with oracle/.
#pragma once
#include <algorithm>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/phs.h"

namespace phs {

// ---- S0: rates and capacities live on an exact fixed-point grid of 2^-20 byte/s (reading R-FX) ----
constexpr int kRateFracBits = 20;
constexpr int kMaxHops = 6;  // longest path: fat tree cross-pod (S2)

// Device-resident flow record, 64 bytes (half a cache line), one per flow.  Everything activation and release
// need sits in the one record, so each costs a single (non-chained) global load: size, timing, the path inline
// (ECMP paths have at most kMaxHops links, -1 padded), the successors and the flow's static link component.
// Successors: a ring flow has at most two, held inline; a longer list lives in succ[] and succ_in[0] is its
// offset into the instance's slice of succ[].
struct FlowRec {
  double bytes;          // flow size
  double start;          // earliest submission time (S4)
  double lat;            // path latency, left-to-right sum over the path's links (S2)
  int32_t path[kMaxHops];  // flow -> link incidence row
  int32_t succ_cnt;      // number of successors
  int32_t succ_in[2];    // succ_cnt <= 2: the successors (instance-relative flow ids, -1 if absent);
                         // succ_cnt > 2: succ_in[0] = offset of the list in succ[]
  int32_t comp;          // static link component of the flow's path (dense id within the unit, in ascending order
                         // of the components' smallest links): two links are in one component iff some chain of
                         // flows of the instance connects them
};
static_assert(sizeof(FlowRec) == 64, "FlowRec must be 64 bytes");

// Descriptor of one simulation unit (device).  A unit is what one CTA / cluster simulates: a whole instance, or --
// when the instance decomposes -- a group of its flows that shares no link and no dependency with the rest (under
// reading R-LZ such a group evolves exactly as it does inside the whole instance).  Flow and link ids inside a
// unit are unit-local and dense.
struct InstDesc {
  int64_t flow_base;  // first entry of the unit in the per-flow arrays (rec, pred_cnt, fmap, ...)
  int64_t link_base;  // first entry of the unit in the per-link arrays (capq, lcomp, linkid)
  int64_t succ_base;  // first entry of the unit's slice of succ[]
  int64_t log_base;   // first row of the unit's event log slice (capacity 2F+2 rows), -1 if disabled
  int64_t pc8_base;   // first byte of the unit's slice of the packed predecessor counters (4-byte aligned)
  int64_t init_base;  // first entry of the unit's slice of the initial-activation list (init_t / init_f)
  int64_t comp_base;  // first entry of the unit in the per-component arrays (cown)
  int32_t n_flows;
  int32_t n_links;
  int32_t n_init;     // flows without predecessors
  int32_t n_comps;    // static link components of the unit (dense ids 0 .. n_comps-1, see FlowRec::comp)
  double lmin;        // lookahead of the unit: the smallest path latency among its flows that have predecessors
                      // (+inf if none has).  A flow released by an event at time t activates no earlier than t + lmin,
                      // so all events in [T0, T0 + lmin) of different components are independent (DESIGN.md sec 4,
                      // "Lookahead windows"); 0 disables the window schedule for the unit.
};

// Per-instance result block (device, read back after a run).
struct InstResult {
  int32_t status;          // PHS_OK, PHS_ECYCLE, or kOverflow (re-run on the cluster path)
  int32_t path;            // 0 = cta, 1 = cluster, 2 = window, 3 = grid
  int64_t n_events;
  int64_t sum_active;
  int64_t sum_par_rounds;
  int32_t max_active;
  int32_t max_pending;
  int32_t max_slots;       // high-water mark of the slot array
  int32_t n_windows;       // lookahead windows of the run (= n_events for a unit that ran one event per iteration)
};
constexpr int32_t kOverflow = 1;  // internal: the CTA path ran out of shared-memory slots
constexpr int32_t kPaused = 2;    // internal: stopped before the first event later than the requested time

// ---- host-side instance tables (built by phs_build.cpp) ----
struct Collective {
  int32_t kind, n_ranks, first_flow, n_flows, steps;
  int32_t chunks = 1;  // pipeline chunks of the chain / tree kinds
  int32_t chain;  // smallest id among the collectives this one is (transitively) chained `after`, else its own id
  std::vector<int32_t> ranks;
  // as submitted: the flows are appended to the instance arrays later (Instance::expanded), on the host threads
  // that build the instance's tables
  double bytes = 0.0, start = 0.0;
  std::vector<int32_t> after;
  std::vector<int32_t> after_flows;  // earlier flows / spans the initial flows additionally wait for, per rank
};

struct Instance {
  uint64_t seed = 0;
  std::vector<double> cap;  // empty: descriptor defaults
  std::vector<int32_t> src, dst;
  std::vector<double> bytes, start, lat;
  std::vector<uint32_t> path_off{0};
  std::vector<int32_t> path;
  std::vector<uint32_t> pred_off{0};
  std::vector<int32_t> pred;
  std::vector<Collective> colls;
  int64_t flow_count = 0;  // flows submitted so far, including those of collectives not expanded yet
  size_t expanded = 0;     // colls[0 .. expanded) have their flows in the arrays above
  int64_t n_flows() const { return flow_count; }
};

// Link numbering and ECMP routing of one topology (S1, S2).
// A user-supplied topology (phs_create_topology_graph): nodes 0 .. n_gpus-1 are the GPUs, the others switches; link i
// is the directed edge from[i] -> to[i].
struct GraphLinks {
  int32_t n_gpus = 0, n_nodes = 0, compute_lanes = 0;
  std::vector<int32_t> from, to;
  std::vector<double> cap, lat;
};

class Fabric {
 public:
  explicit Fabric(const phs_topology_desc &d);
  explicit Fabric(GraphLinks g);  // shortest-path ECMP over the link list (S8)
  static phs_status validate_graph(const GraphLinks &g, std::string *why);
  // is there a route of at most kMaxHops links?  (always, on the preset topologies)
  bool routable(int32_t src, int32_t dst) const;
  static phs_status validate(const phs_topology_desc &d, std::string *why);
  int32_t n_gpus() const { return gpus_; }
  int32_t n_links() const { return links_; }
  double default_capacity(int32_t link) const;
  double latency(int32_t link) const {  // engine links: 0
    return link >= net_links_ ? 0.0 : graph_ ? g_.lat[(size_t)link] : d_.hop_latency_s;
  }
  int32_t n_net_links() const { return net_links_; }
  int32_t compute_lanes() const { return d_.compute_lanes; }
  // writes the links of (src -> dst) for connection key `conn` into out[0..kMaxHops), returns the hop count
  int route(uint64_t seed, int32_t src, int32_t dst, int32_t conn, int32_t *out) const;

 private:
  phs_topology_desc d_;
  int32_t gpus_, links_, net_links_, tier1_base_, tier2_base_;
  bool graph_ = false;
  GraphLinks g_;
  std::vector<int32_t> out_off_, out_link_;  // out-links of every node, ascending link id
  std::vector<int16_t> hops_;                // [gpu][node] links on a shortest path node -> gpu, -1 = unreachable
};

uint64_t splitmix64_step(uint64_t x);

// Appends the flows of every collective that was submitted but not expanded yet (S3); idempotent.
void expand_pending(const Fabric &fab, Instance &inst);

// Appends flows / collectives to an instance (S3).  Return PHS_OK or an error with *why set.  append_collective
// validates and records the collective; its flows appear with the next expand_pending.
phs_status append_collective(const Fabric &fab, Instance &inst, int32_t kind, const int32_t *ranks, int32_t n_ranks,
                             double bytes, double start, const int32_t *after, int32_t n_after,
                             const int64_t *after_flows, int32_t n_after_flows, int32_t chunks, std::string *why,
                             bool checked = false);
phs_status append_spans(const Fabric &fab, Instance &inst, int64_t n, const int32_t *gpu, const int32_t *lane,
                        const double *duration, const double *start, const int64_t *dep_off, const int64_t *dep_ids,
                        std::string *why);
phs_status append_flows(const Fabric &fab, Instance &inst, int64_t n, const int32_t *src, const int32_t *dst,
                        const double *bytes, const double *start, const int64_t *dep_off, const int64_t *dep_ids,
                        const int32_t *conn_id, std::string *why);

}  // namespace phs
