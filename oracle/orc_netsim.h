/*
 * orc_netsim.h -- CPU ORACLE for the flow-level network simulator (netsim) of
 * Phantora (arxiv 2505.01616).  TEST INFRASTRUCTURE ONLY.
 *
 * This is a plain, slow, single-threaded, obviously-correct C restatement of
 * what the hot path computes.  It shares no code with the CUDA library
 * (paper_2505_01616_b200/csrc) and is never used by the product path: only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load it.
 *
 * Passages followed (PAPER.md line numbers):
 *   L98  (sec 4.1)  netsim: topology config (port bandwidth, interconnection,
 *                   multipath routing / load balancing); throughput of flows at
 *                   each time = max-min fairness; collective patterns.
 *   L104 (sec 4.1)  ring all-reduce; flows submitted with timestamps; output =
 *                   completion time of each flow.
 *   L128 (sec 4.2)  between neighbouring events flows have stable throughput.
 *   L165 (sec 5)    per-flow fairness; iterative water-filling; each iteration
 *                   identifies THE bottleneck link and adjusts flow rates.
 *   L308 (sec 7)    a flow immediately reaches its fair share.
 * Everything the paper leaves open follows the readings S0-S6 / Q1-Q18 of
 * SURVEY.md sec 8(c), restated in DESIGN.md ("Readings").  One reading is the
 * builder's own and is listed there as R-FX: rates, capacities and fair shares
 * are held in exact 64-bit fixed point (quantum 2^-20 byte/s), so that the
 * water-filling result does not depend on the order in which capacity debits
 * are applied.  Time and byte arithmetic is IEEE binary64 without contraction.
 * A second builder's reading, R-LZ (from L128 "between neighboring events, network flows are assumed to have
 * stable throughput" and L167, where a flow's history is "a few floating point numbers" per throughput
 * change): a flow's remaining bytes are settled only when ITS rate changes, so its completion time is a
 * function of its own rate history and not of unrelated events elsewhere in the network.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): P1 lone flow, P2 uniform
 * ring, P3 max-plus ring recurrence (cfg0), P4 bottleneck certificate, P5
 * brute-force lexicographic max-min, P6 processor sharing, P7 parking lot,
 * P8 uniform all-to-all, P9 invariances, naive == fast mode.
 * "parity unpinned": the ECMP hash VALUE (S2) -- the paper gives none; it is
 * pinned only against published SplitMix64 outputs and by balance statistics.
 */
#ifndef ORC_NETSIM_H
#define ORC_NETSIM_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_sim orc_sim;

enum { ORC_OK = 0, ORC_EINVAL = -1, ORC_ENOMEM = -2, ORC_ECYCLE = -4, ORC_ESTATE = -5, ORC_ERANGE = -6 };
enum { ORC_TOPO_SINGLE = 0, ORC_TOPO_LEAF_SPINE = 1, ORC_TOPO_FAT_TREE = 2, ORC_TOPO_GRAPH = 3 };
enum { ORC_ALLREDUCE_RING = 0, ORC_ALLGATHER_RING = 1, ORC_REDUCESCATTER_RING = 2, ORC_ALLTOALL = 3,
       /* NEXT-3: pipelined chain broadcast / reduce, binary-tree all-reduce; see orc_add_collective_ex */
       ORC_BROADCAST_CHAIN = 4, ORC_REDUCE_CHAIN = 5, ORC_ALLREDUCE_TREE = 6 };
enum { ORC_MODE_NAIVE = 0, ORC_MODE_FAST = 1 };
/* orc_run_ex flags: the two readings of SURVEY.md 8(c) that DESIGN.md sec 2 replaced, kept for comparison */
enum { ORC_FLAG_SETTLE_EVERY_EVENT = 1, /* S4.4 as written: every ACTIVE flow is debited at every event (not R-LZ) */
       ORC_FLAG_F64_SHARES = 2 };       /* S5 as written: binary64 cap_rem / share (not R-FX); naive mode only      */

typedef struct {
  int32_t kind, n_hosts, gpus_per_host;
  double nvlink_Bps, nic_Bps, fabric_Bps, hop_latency_s; /* per direction */
  int32_t n_leaves, n_spines, uplinks_per_leaf_spine;    /* leaf-spine */
  int32_t k, agg_uplinks;                                /* fat tree */
  int32_t compute_lanes;                                 /* NEXT-2: compute engines per GPU (0 = none), see orc_add_spans */
} orc_topology_desc;

typedef struct {
  double t;             /* time the clock moved to in this loop iteration */
  int32_t n_completed;  /* flows that completed at t */
  int32_t n_activated;  /* flows activated at the start of the iteration */
  int32_t n_rounds;     /* water-filling iterations of this iteration's solve */
  int32_t first_bneck;  /* bottleneck link of the first iteration, -1 if none */
} orc_event;

/* One simulation instance.  `seed` is the instance's ECMP seed. */
int32_t orc_create_topology(const orc_topology_desc *d, uint64_t seed, orc_sim **out);
/* NEXT-4, user-supplied topology ("netsim takes a cluster topology configuration as input ... switch
 * port bandwidth, cluster interconnection, multipath routing").  Reading S8: nodes 0..n_gpus-1 are the
 * GPUs, the others switches; link i is the directed edge link_from[i] -> link_to[i] with its own capacity (byte/s)
 * and latency (s); link ids are the caller's.  Routing = shortest paths by hop count with seeded ECMP: at node u
 * the candidates are the out-links (u -> v) with dist(v, dst) = dist(u, dst) - 1, in ascending link id, and hop k
 * (k = 0, 1, ...) takes candidate mix(H ^ (k + 1)) mod #candidates, H = the S2 hash of (seed, src, dst, conn).
 * Paths longer than 6 links and unreachable pairs are refused when the flow is added. */
int32_t orc_create_topology_graph(int32_t n_gpus, int32_t n_nodes, int32_t n_links, const int32_t *link_from,
                                  const int32_t *link_to, const double *cap_Bps, const double *latency_s,
                                  int32_t compute_lanes, uint64_t seed, orc_sim **out);
void orc_destroy(orc_sim *s);
int32_t orc_num_links(const orc_sim *s, int32_t *out);
int32_t orc_set_link_capacities(orc_sim *s, const double *cap_Bps);
int32_t orc_get_link_capacities(const orc_sim *s, double *cap_Bps);
int32_t orc_add_collective(orc_sim *s, int32_t kind, const int32_t *ranks, int32_t n_ranks, double bytes,
                           double start_time_s, const int32_t *after, int32_t n_after, int32_t *out_coll_id);
/* the same with `chunks` pipeline chunks (chain and tree kinds; 1 for the others) */
int32_t orc_add_collective_ex(orc_sim *s, int32_t kind, const int32_t *ranks, int32_t n_ranks, double bytes,
                              double start_time_s, const int32_t *after, int32_t n_after, int32_t chunks,
                              int32_t *out_coll_id);
int32_t orc_add_flows(orc_sim *s, int64_t n, const int32_t *src, const int32_t *dst, const double *bytes,
                      const double *start_time_s, const int64_t *dep_off, const int64_t *dep_flow_ids,
                      const int32_t *conn_id, int64_t *out_first_flow_id);
/* NEXT-2, compute spans (PAPER.md L84 / L94 / L106: the event queue holds compute and communication spans with
 * explicit dependencies; L206 / Fig. 7: computation overlaps communication).  A span is a DAG node of fixed length
 * bound to a compute engine ("lane") of a GPU.  Reading S7: every GPU has `compute_lanes` engine links,
 * numbered after all network links (id = n_network_links + gpu * compute_lanes + lane), of capacity 2^32 work
 * units / s and latency 0; a span of d seconds is a flow of d * 2^32 units over its engine link (src = dst = gpu).
 * Alone on its lane it runs at 2^32 units / s, so it finishes at exactly t_act + d (scaling by a power of two is
 * exact); spans that overlap on one lane share it max-min fairly (processor sharing).  Spans take flow ids like
 * raw flows, depend on earlier flows / spans, and flows may depend on them. */
int32_t orc_add_spans(orc_sim *s, int64_t n, const int32_t *gpu, const int32_t *lane, const double *duration_s,
                      const double *start_time_s, const int64_t *dep_off, const int64_t *dep_flow_ids,
                      int64_t *out_first_flow_id);
/* orc_add_collective_ex plus flow-level predecessors: every flow of the collective that has no predecessor inside it
 * and is sent by rank rho additionally waits for each listed EARLIER flow or span whose source or destination is rho */
int32_t orc_add_collective_full(orc_sim *s, int32_t kind, const int32_t *ranks, int32_t n_ranks, double bytes,
                                double start_time_s, const int32_t *after, int32_t n_after, const int64_t *after_flows,
                                int32_t n_after_flows, int32_t chunks, int32_t *out_coll_id);
/* trace != 0 additionally records, for every loop iteration, the active flows and their rates */
int32_t orc_run(orc_sim *s, int32_t mode, int32_t trace);
/* same, but stops before the first event later than t_stop ("advancing the simulation ... up to a
 * specified time"); unfinished flows keep t_done = NaN and bneck = -1 */
int32_t orc_run_until(orc_sim *s, int32_t mode, int32_t trace, double t_stop);
/* NEXT-1, time rollback (sec 4.2, L167 sec 5).  orc_run / orc_run_until may be called again: a
 * call CONTINUES from the events simulated so far (a larger stop time advances "up to a specified time", L167), after
 * rebuilding the simulator state from the per-flow throughput history (L128).  Submissions after a run
 * (orc_add_flows / orc_add_collective* / orc_add_spans) and orc_update_flow_start roll back to the (earlier) start
 * time involved; orc_rollback does it explicitly; orc_gc drops history that no later rollback to a time >= T needs
 * (L130) -- a rollback below the watermark then fails with ORC_EINVAL. */
int32_t orc_rollback(orc_sim *s, double T);
int32_t orc_update_flow_start(orc_sim *s, int64_t flow, double start_time_s);
int32_t orc_gc(orc_sim *s, double T);
/* the same with `flags` (see above); flags = 0 is orc_run_until */
int32_t orc_run_ex(orc_sim *s, int32_t mode, int32_t trace, double t_stop, int32_t flags);
/* S4.4 / Q11 settle step on its own: max(rem - rate * dt, 0) with mul, sub, clamp in that order */
double orc_settle(double rem, double rate_Bps, double dt);
int32_t orc_num_flows(const orc_sim *s, int64_t *out);
int32_t orc_get_completion_times(const orc_sim *s, double *out, int64_t n);
int32_t orc_get_bottlenecks(const orc_sim *s, int32_t *out, int64_t n);
int32_t orc_num_collectives(const orc_sim *s, int32_t *out);
int32_t orc_get_collective_times(const orc_sim *s, double *out, int32_t n);
int32_t orc_num_events(const orc_sim *s, int64_t *out);
int32_t orc_get_event_log(const orc_sim *s, orc_event *out, int64_t cap, int64_t *n_events);
int32_t orc_get_paths(const orc_sim *s, int64_t *off /*[F+1]*/, int32_t *links, int64_t cap);
int32_t orc_num_path_entries(const orc_sim *s, int64_t *out);
int32_t orc_get_flow_endpoints(const orc_sim *s, int32_t *src, int32_t *dst, double *bytes, double *lat, int64_t n);
int32_t orc_get_preds(const orc_sim *s, int64_t *off /*[F+1]*/, int32_t *preds, int64_t cap, int64_t *n_entries);
/* work counters of the last run: [0] sum over events of A (active flows), [1] sum A*h (path entries of
 * active flows), [2] sum of water-filling iterations R, [3] sum over events of Lambda_act*R,
 * [4] sum Lambda_act, [5] completions, [6] events */
int32_t orc_get_work_counters(const orc_sim *s, double *out7);
/* throughput history (PAPER.md L128 / L167; reading R-LZ): one record (flow, time, new rate in byte/s) per rate
 * change of a flow, in the order the event loop produced them (chronological; within an event in the order of
 * the active list).  A flow's records partition its life into intervals of constant throughput:
 * bytes = sum rate_i * (t_{i+1} - t_i) with the completion time closing the last interval. */
int32_t orc_history_size(const orc_sim *s, int64_t *n_records);
int32_t orc_get_history(const orc_sim *s, int32_t *flow, double *t, double *rate_Bps, int64_t cap);
/* trace access (valid after orc_run(..., trace=1)) */
int32_t orc_trace_size(const orc_sim *s, int64_t *n_rows);
int32_t orc_get_trace(const orc_sim *s, int64_t *event_idx, int32_t *flow, double *rate_Bps, double *t0, double *t1,
                      int64_t cap);

/* Stand-alone max-min progressive filling (S5) on an explicit instance: flows given as CSR paths over
 * n_links links.  rate_Bps[f], bneck[f] out; *n_rounds, *first_bneck out.  mode as in orc_run. */
int32_t orc_maxmin(int32_t n_links, const double *cap_Bps, int32_t n_flows, const int64_t *path_off,
                   const int32_t *path, int32_t mode, double *rate_Bps, int32_t *bneck, int32_t *n_rounds,
                   int32_t *first_bneck);
/* SplitMix64 step used by the ECMP hash (S2) */
uint64_t orc_mix64(uint64_t x);

#ifdef __cplusplus
}
#endif
#endif
