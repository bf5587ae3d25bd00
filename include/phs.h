/*
 * phs.h -- C-ABI of libphs: a B200-native (sm_100a) batched flow-level network simulator, the netsim hot
 * path of Phantora (arxiv 2505.01616).  All entry points are extern "C", take plain pointers and sizes and
 * never throw.  Pointers are HOST pointers unless the argument says "device".
 *
 * What the calls mean, by passage of the paper (PAPER.md line numbers; DESIGN.md gives the readings S0-S6):
 *   phs_create_topology      L98  "netsim takes a cluster topology configuration as input ... switch port
 *                                  bandwidth, cluster interconnection, multipath routing and load balancing"
 *   phs_add_collective       L98/L104 "we implement the communication patterns of different collective
 *                                  operations ... all reduce using a ring-based approach"
 *   phs_add_flows            L104 "submits the corresponding data transfer flows to netsim with the
 *                                  appropriate timestamps"
 *   phs_run                  L165 max-min fair allocation by iterative water-filling; L128 piecewise-constant
 *                                  throughput between events; L308 flows reach their fair share at once
 *   phs_get_completion_times L104 "computes the completion time of each flow"
 *   phs_get_bottlenecks, phs_get_event_log   L165 "the simulator identifies the bottleneck link" (per flow: the link
 *                                  that froze it in its last solve; per event: iterations and first bottleneck)
 *   phs_get_collective_times L104 the collective completes when its last flow does
 *   phs_set_link_capacities*, phs_get_paths, phs_get_preds, phs_get_flow_table   L98 port bandwidth, routing; L104 the
 *                                  flow patterns of the collectives, as tables for integer parity
 *   phs_run_until, phs_update_flow_start, phs_rollback, phs_gc   L124-130, L167 (time rollback, advancing up to a time)
 *   phs_enable_history / phs_get_flow_history   L128, L167 (piecewise-constant throughput, a few numbers per change)
 *   phs_add_spans            L84 / L94 / L106 / L206 (compute spans in the event DAG)
 *   phs_create_topology_graph, phs_set_devices   L98 (topology configuration as input); SURVEY.md 8(e)
 *
 * Ownership: the caller owns every array it passes; the library copies inputs before returning.  Outputs go
 * to caller-provided buffers.  Ids are dense and assigned in call order: flow ids per instance start at 0, a
 * collective's flows are contiguous (ring: step-major, then ring index; all-to-all: row-major without the
 * diagonal).  A handle is not thread-safe; distinct handles are independent.
 *
 * Errors: every call returns a phs_status; <0 is an error and phs_last_error() gives a thread-local message.
 * The library has NO CPU fallback: phs_finalize / phs_run return PHS_ECUDA when no CUDA device is usable.
 */
#ifndef PHS_H
#define PHS_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct phs_sim phs_sim; /* opaque; owned by the library; freed by phs_destroy */
typedef int32_t phs_status;
enum {
  PHS_OK = 0,
  PHS_EINVAL = -1, /* bad argument: null pointer, bytes <= 0 or NaN, src == dst, rank out of range, ...   */
  PHS_ENOMEM = -2, /* host or device allocation failed                                                    */
  PHS_ECUDA = -3,  /* CUDA failure (no device, launch error, ...); message holds the CUDA string          */
  PHS_ECYCLE = -4, /* flows left WAITING when nothing is active or pending (dependency never satisfied)   */
  PHS_ESTATE = -5, /* call not valid in this state (adding after phs_finalize, reading before phs_run)    */
  PHS_ERANGE = -6  /* size limit exceeded (>= 2^31 flows per instance, capacity < #flows quanta, ...)     */
};
typedef enum { PHS_TOPO_SINGLE = 0, PHS_TOPO_LEAF_SPINE = 1, PHS_TOPO_FAT_TREE = 2 } phs_topo_kind;
typedef enum {
  PHS_ALLREDUCE_RING = 0,     /* 2(N-1) steps of N flows, chunk = bytes/N      */
  PHS_ALLGATHER_RING = 1,     /* (N-1) steps; bytes = total gathered size      */
  PHS_REDUCESCATTER_RING = 2, /* (N-1) steps; bytes = total input size         */
  PHS_ALLTOALL = 3,           /* N(N-1) concurrent flows of bytes/N            */
  /* further collective algorithms ("the communication patterns of different collective operations"),
   * with C = `chunks` pipeline chunks of bytes/C (phs_add_collective_ex): */
  PHS_BROADCAST_CHAIN = 4,    /* root ranks[0]; hop i: ranks[i] -> ranks[i+1]; C(N-1) flows, chunk-major        */
  PHS_REDUCE_CHAIN = 5,       /* towards the root: hop i: ranks[N-1-i] -> ranks[N-2-i]                           */
  PHS_ALLREDUCE_TREE = 6      /* binary tree in heap order over the ranks: per chunk N-1 up flows (child ->      */
                              /* parent), then N-1 down flows; 2C(N-1) flows                                      */
} phs_coll_kind;

/* Topology descriptor (S1).  GPU g = host*gpus_per_host + local.  Every physical link is two
 * directed links with the same capacity; capacities are byte/s PER DIRECTION; every link adds hop_latency_s. */
typedef struct {
  int32_t kind;                 /* phs_topo_kind                                                          */
  int32_t n_hosts, gpus_per_host;
  double nvlink_Bps;            /* GPU <-> its host's NVSwitch                                            */
  double nic_Bps;               /* GPU <-> first-tier switch (one NIC per GPU)                            */
  double fabric_Bps;            /* switch <-> switch                                                      */
  double hop_latency_s;
  int32_t n_leaves, n_spines, uplinks_per_leaf_spine; /* leaf-spine: hosts in contiguous blocks per leaf  */
  int32_t k, agg_uplinks;       /* fat tree: k pods, k/2 edge (= hosts) and k/2 agg switches per pod,
                                   gpus_per_host = k/2, n_hosts = k*k/2; agg_uplinks per agg switch       */
  int32_t compute_lanes;        /* compute engines per GPU for phs_add_spans (0 = none): engine links are
                                   numbered after all network links, n_network_links + gpu * compute_lanes + lane,
                                   capacity 2^32 work units / s, latency 0                                 */
} phs_topology_desc;

/* One row of the event log (S6/O4): one loop iteration = one distinct time. */
typedef struct {
  double t;            /* time the clock moved to                                                         */
  int32_t n_completed; /* flows that completed at t                                                       */
  int32_t n_activated; /* flows activated at the start of the iteration                                   */
  int32_t n_rounds;    /* bottleneck links frozen by this iteration's max-min solve                       */
  int32_t first_bneck; /* link with the smallest fair share at the start of the solve, -1 if none active  */
} phs_event;

/* Per-run work counters, summed over the simulation units of the last phs_run (an instance is one unit, or --
 * with decomposition -- several independent ones; events that coincide in time in different units count once
 * per unit). */
typedef struct {
  int64_t n_events;      /* loop iterations                                                               */
  int64_t n_flow_events; /* activations + completions = 2 * flows                                         */
  int64_t sum_active;    /* sum over events of active flows                                               */
  int64_t sum_par_rounds;/* sum over events of parallel filling rounds executed by the kernels            */
  int64_t n_kernel_launches; /* kernels launched by the last phs_run                                      */
  int64_t h2d_bytes;     /* bytes phs_finalize copied to the device                                       */
  int32_t max_active;    /* largest number of simultaneously ACTIVE flows in one instance                 */
  int32_t max_slots;     /* largest number of state slots (PENDING + ACTIVE flows) one instance ever used */
  int32_t cluster_size;  /* CTAs per cluster of the cluster path in the last run (0: path not used)            */
  int32_t clusters_resident; /* clusters of that size the device keeps resident at once                        */
  int32_t resumed_units; /* units the last phs_run_until continued from their parked state (0: started at t = 0) */
  int32_t window_gang;   /* CTAs per unit of the window path in the last run (largest gang; 0: path not used)     */
  double main_kernel_ms; /* device time of the simulation kernel(s) of the last phs_run (CUDA events on   */
                         /* the run's stream), excluding the result copies                                */
  int32_t grid_ctas;     /* CTAs of the cooperative launch of the grid path in the last run (0: path not used)   */
  int32_t pad_;
  double resumed_from_s; /* simulated time of the parked state / snapshot the last run continued from (0: it      */
                         /* started at t = 0)                                                                   */
  int64_t n_windows;     /* lookahead windows executed (phs_set_windows); = n_events where the window schedule  */
                         /* is off.  n_events then counts window ITERATIONS: one iteration advances every       */
                         /* component that has an event inside the window by one event                          */
} phs_counters;

/* Creates `batch` independent instances of one topology.  Instance i routes with ECMP seed `seed + i`.
 * Host-only; never touches the GPU. */
phs_status phs_create_topology(const phs_topology_desc *desc, uint64_t seed, int32_t batch, phs_sim **out);
/* User-supplied topology ("netsim takes a cluster topology configuration as input ... switch port
 * bandwidth, cluster interconnection, multipath routing and load balancing strategies").  Nodes 0 .. n_gpus-1 are the
 * GPUs, the others switches; link i (its id in every output) is the directed edge link_from[i] -> link_to[i] with
 * capacity cap_Bps[i] and latency latency_s[i]; compute engine links (compute_lanes per GPU) follow.  Routing:
 * shortest paths by hop count with seeded ECMP -- at a node the candidates are the out-links that lead one hop closer
 * to the destination, in ascending link id, and hop k takes candidate mix(H ^ (k+1)) mod #candidates, H the hash of
 * (seed, src, dst, connection) of the preset topologies.  Flows between GPUs without a route of at most 6 links are
 * refused (PHS_EINVAL) when they are added. */
phs_status phs_create_topology_graph(int32_t n_gpus, int32_t n_nodes, int32_t n_links, const int32_t *link_from,
                                     const int32_t *link_to, const double *cap_Bps, const double *latency_s,
                                     int32_t compute_lanes, uint64_t seed, int32_t batch, phs_sim **out);
void phs_destroy(phs_sim *sim);
phs_status phs_num_links(const phs_sim *sim, int32_t *out);
phs_status phs_batch(const phs_sim *sim, int32_t *out);

/* Overrides the capacities (byte/s, [n_links], S1 numbering) of one instance (-1: all). */
phs_status phs_set_link_capacities(phs_sim *sim, int32_t instance, const double *cap_Bps);
phs_status phs_get_link_capacities(const phs_sim *sim, int32_t instance, double *cap_Bps);
/* The same for every instance at once (the parameter sweep of BASELINE.json configs[3]): cap_Bps is a host array
 * [batch][n_links], row i for instance i; the library copies it.  PHS_EINVAL (nothing changed) if any entry is
 * outside (0, 2^42) byte/s; PHS_ESTATE after phs_finalize. */
phs_status phs_set_link_capacities_batch(phs_sim *sim, const double *cap_Bps);

/* Adds one collective over `ranks` (ring order) to `instance` (-1: every instance).  `after_coll_ids`
 * (nullable) chains it per rank behind earlier collectives of the same instance (S3).
 * out_coll_id (nullable) receives the collective's id.  The call validates its arguments, copies them and assigns
 * the flow ids at once (phs_num_flows counts them); the flows themselves -- routes and DAG edges, PAPER.md L98 / L104 --
 * are materialised by the next phs_add_flows on that instance, a table getter or phs_finalize. */
phs_status phs_add_collective(phs_sim *sim, int32_t instance, int32_t kind, const int32_t *ranks, int32_t n_ranks,
                              double bytes, double start_time_s, const int32_t *after_coll_ids, int32_t n_after,
                              int32_t *out_coll_id);
/* The same with `chunks` >= 1 pipeline chunks for the chain and tree kinds (must be 1 for the ring kinds and the
 * all-to-all).  A flow of chunk c on a hop waits for the previous hop's flow of chunk c (the data is there) and for
 * the same hop's flow of chunk c-1 (FIFO per connection); S3 gives ids and dependencies.  `start_time_s` and
 * the `after` edges apply to every flow without a predecessor inside the collective; as an `after` target such a
 * collective contributes, per rank, the flows of its last chunk the rank sends or receives. */
phs_status phs_add_collective_ex(phs_sim *sim, int32_t instance, int32_t kind, const int32_t *ranks, int32_t n_ranks,
                                 double bytes, double start_time_s, const int32_t *after_coll_ids, int32_t n_after,
                                 int32_t chunks, int32_t *out_coll_id);
/* Same collective on EVERY instance with per-instance sizes / start times: bytes[batch], start_time_s[batch]
 * (nullable = 0). */
phs_status phs_add_collective_batch(phs_sim *sim, int32_t kind, const int32_t *ranks, int32_t n_ranks,
                                    const double *bytes, const double *start_time_s, const int32_t *after_coll_ids,
                                    int32_t n_after, int32_t *out_coll_id);
/* Adds n raw flows (after phs_finalize: a late submission, see phs_update_flow_start).  start_time_s nullable (= 0).  dep_off[n+1]/dep_flow_ids (nullable) list, per flow, ids of
 * EARLIER flows of the same instance that must complete first.  conn_id (nullable = the flow's id) keys ECMP. */
phs_status phs_add_flows(phs_sim *sim, int32_t instance, int64_t n, const int32_t *src, const int32_t *dst,
                         const double *bytes, const double *start_time_s, const int64_t *dep_off,
                         const int64_t *dep_flow_ids, const int32_t *conn_id, int64_t *out_first_flow_id);

/* Compute spans (PAPER.md L84 / L94 / L106: the event queue holds compute and communication spans with explicit
 * dependencies; L206 / Fig. 7: computation overlapping communication).  A span is a DAG node of fixed length bound to
 * a compute lane of a GPU: a flow of duration_s * 2^32 work units over that lane's engine link (src = dst = gpu).
 * Alone on its lane it finishes at exactly t_act + duration_s; spans that overlap on one lane share it max-min fairly.
 * Spans take flow ids like raw flows (out_first_flow_id), may depend on earlier flows / spans (dep_off / dep_flow_ids
 * as in phs_add_flows) and may be depended upon; their "bottleneck" is the engine link.  lane nullable (= 0),
 * start_time_s nullable (= 0); duration in (0, 2^20) s.  Needs compute_lanes > 0 in the topology descriptor. */
phs_status phs_add_spans(phs_sim *sim, int32_t instance, int64_t n, const int32_t *gpu, const int32_t *lane,
                         const double *duration_s, const double *start_time_s, const int64_t *dep_off,
                         const int64_t *dep_flow_ids, int64_t *out_first_flow_id);
/* phs_add_collective_ex plus flow-level predecessors: every flow of the collective that has no predecessor inside it
 * and is sent by rank rho additionally waits for each listed EARLIER flow or span whose source or destination is rho
 * (a span's is its GPU): "the all-reduce of a layer's gradients starts when that rank's backward kernel is done". */
phs_status phs_add_collective_full(phs_sim *sim, int32_t instance, int32_t kind, const int32_t *ranks, int32_t n_ranks,
                                   double bytes, double start_time_s, const int32_t *after_coll_ids, int32_t n_after,
                                   const int64_t *after_flow_ids, int32_t n_after_flows, int32_t chunks,
                                   int32_t *out_coll_id);

/* Event log on/off (default off) for subsequent runs; must precede phs_finalize. */
phs_status phs_enable_event_log(phs_sim *sim, int32_t enable);

/* Batch-scheduler policy; must precede phs_finalize.  path: 0 = automatic (units whose events
 * are dense in simulated time run the lookahead-window schedule on a gang of CTAs; of the others, one CTA per
 * simulation unit with all state in its shared memory when it fits, else one thread-block cluster per unit with the
 * state spread over the shared memory of its CTAs; a unit that fits no cluster is simulated by the whole grid with
 * its state in global memory), 1 = CTA path, 2 = cluster path for every unit, 3 = window path for every unit that
 * can run there (positive latency, no event log, no history), 4 = grid path for every unit (no event log).  cta_slots > 0 caps the CTA
 * path's shared-memory slot count (flows PENDING or ACTIVE at once per unit); a unit that exceeds it is re-run on
 * the cluster path.  With path = 3, cta_slots is instead the smallest gang (CTAs per unit: 1, 2, 4, 8, 16) to use
 * for units that have enough components. */
phs_status phs_set_scheduler(phs_sim *sim, int32_t path, int32_t cta_slots);

/* Decomposition (default on).  An instance whose flows fall into groups that share no link and no dependency is
 * simulated as independent units, one CTA / cluster each; under reading R-LZ the results are
 * bit-identical to simulating the instance as a whole.  Off: one unit per instance.  The event log needs the
 * instance-wide event sequence, so enabling it turns decomposition off.  Must precede phs_finalize. */
phs_status phs_set_decomposition(phs_sim *sim, int32_t enable);

/* Lookahead windows (default on).  A flow released by an event at time t starts no earlier than t + L, L = the
 * smallest path latency of the unit's dependent flows, and static link components influence each other only through
 * such releases; so the events of different components inside [T0, T0 + L) are independent and one loop iteration
 * of the kernels advances all of them, each at its own time.  Results are bit-identical to the one-event-per-
 * iteration schedule (reading R-LZ).  Units with zero latency, the event log or the throughput history
 * always run one event per iteration.  Must precede phs_finalize. */
phs_status phs_set_windows(phs_sim *sim, int32_t enable);

/* Multi-GPU (batches shard naturally, a single instance does not).  Binds the handle to n CUDA
 * devices of this process: phs_finalize cuts the batch into n contiguous blocks of instances (instance i keeps its ECMP
 * seed `seed + i`) and builds block k's tables on device_ids[k]; phs_run / phs_run_until simulate all blocks at once
 * (one host thread per device, each device's default stream: the cuda_stream argument is ignored); result getters go
 * to the device that holds the instance, and an out_is_device buffer must live there.  No data-path collective
 * exists or is needed.  A device may be listed more than once.  phs_get_all_* return host arrays only, and late
 * submissions (after phs_finalize) are not supported on such a handle (PHS_ESTATE).  Must precede phs_finalize. */
phs_status phs_set_devices(phs_sim *sim, int32_t n, const int32_t *device_ids);
/* Device that holds `instance` after phs_finalize (the current device for a single-device handle). */
phs_status phs_instance_device(const phs_sim *sim, int32_t instance, int32_t *out);

/* Throughput history ("between neighboring events, network flows are assumed to have stable
 * throughput"; L167: a flow's history is a few floating point numbers per throughput change, from which a time
 * rollback reconstructs the state).  When enabled, every rate change of every flow is recorded as (time, new rate);
 * a flow's records partition its life into intervals of constant throughput that end at its completion time.
 * `max_records` bounds the records of one run over the whole batch; a run that produces more fails with PHS_ERANGE
 * (the message names the number needed).  Must precede phs_finalize. */
phs_status phs_enable_history(phs_sim *sim, int64_t max_records);
/* History of one instance after phs_run, as CSR over its flows: off[F+1], then per record the time and the new
 * rate in byte/s, chronological per flow.  n_records (nullable) receives the record count; t / rate_Bps may be
 * null to query it; cap = capacity of t and rate_Bps. */
phs_status phs_get_flow_history(const phs_sim *sim, int32_t instance, int64_t *off, double *t, double *rate_Bps,
                                int64_t cap, int64_t *n_records);

/* Builds the device-resident tables (flow records, flow->link CSR, successor CSR, capacities) and copies them
 * to the current CUDA device on `cuda_stream` (cudaStream_t; NULL = default stream).  After this call the
 * instance set is frozen (adds return PHS_ESTATE).  phs_run calls it implicitly if needed. */
phs_status phs_finalize(phs_sim *sim, void *cuda_stream);
/* Runs every instance to completion on the GPU (all steps of the hot path in CUDA kernels) and waits for the
 * result status.  May be called repeatedly: after a complete run it starts again from t = 0; after a phs_run_until
 * that stopped early it continues from the parked state.  After an error return the handle holds no results (getters
 * return PHS_ESTATE) and the next run starts from t = 0. */
phs_status phs_run(phs_sim *sim, void *cuda_stream);
/* PAPER.md L167 "advancing the simulation ... up to a specified time": like phs_run, but stops before the first
 * event later than t_stop_s.  Flows that complete later report completion time NaN and bottleneck -1, a collective
 * with such flows reports NaN; event log and throughput history hold what happened up to t_stop_s.  A later call
 * with a larger time continues: a unit that stopped keeps a copy of its on-chip state in global memory and resumes
 * from it; if the time goes backwards everything starts again from t = 0 -- the simulation is deterministic, so
 * the results are the same either way. */
phs_status phs_run_until(phs_sim *sim, double t_stop_s, void *cuda_stream);

/* phs_run without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it).  Same computation as phs_run (PAPER.md L165 water-filling, L128 / L308 event
 * loop, L104 completion times), every unit simulated by the whole grid (the grid path of phs_set_scheduler), but the
 * kernel's scratch -- per-flow and per-link state, and the unit list -- is a fixed __device__ array of
 * PHS_STATIC_SCRATCH_BYTES inside the library (every GPU that loads libphs holds it until the process exits) instead of
 * memory from cudaMalloc.  The call makes no cudaMalloc / cudaFree / cudaHostAlloc and calls no allocating routine; it
 * enqueues on `cuda_stream` and waits for the status, like phs_run.
 *   inputs   the handle: it must be finalized (phs_finalize builds the device tables -- call it at set-up), bound to
 *            one device (the current one, or the one of phs_set_devices), without event log and throughput history.
 *   outputs  t_done_dev[n], bneck_dev[n]: DEVICE arrays of the caller on the handle's device, n = phs_total_flows,
 *            all instances concatenated in instance order (either may be NULL).  The handle holds the same results:
 *            the phs_get_* calls work after it as after phs_run.
 *   limits   PHS_ERANGE (nothing ran; the message names the sizes) if the handle has more than PHS_STATIC_MAX_UNITS
 *            simulation units, or if its largest unit needs more than PHS_STATIC_SCRATCH_BYTES - 4 * PHS_STATIC_MAX_UNITS
 *            bytes of state: 40 bytes per flow + 64 per link + 1 KiB, i.e. about 200,000 flows in one unit.
 *   sharing  every call on a device uses the one array, which keeps the contents of the last call; the kernel
 *            initialises all of it that it reads, so nothing carries over.  Two calls that overlap on one GPU (two
 *            streams, two threads, two handles) race: serialise them.
 * PHS_ESTATE if the handle is not finalized, has several devices, or has the event log / history enabled. */
#define PHS_STATIC_SCRATCH_BYTES (8u << 20)
#define PHS_STATIC_MAX_UNITS 4096
phs_status phs_run_static(phs_sim *sim, void *cuda_stream, double *t_done_dev, int32_t *bneck_dev, int64_t n);

/* Time rollback (sec 4.2 "the network simulator rolls back to T2 and adds a flow starting at T2",
 * Fig. 4; L167 sec 5: "one for updating the start time of an existing flow, and another for advancing the simulation
 * ... up to a specified time").
 *   phs_set_snapshots   every phs_run_until that stops at a time keeps the parked state of that time (on-chip state
 *                       of every unit + outstanding-predecessor counters); the newest `n` are held.  A later run that
 *                       must go back in time continues from the newest usable snapshot instead of t = 0.
 *   phs_update_flow_start  changes the start time of a flow after phs_finalize.  The start time acts through
 *                       t_act = max(start, release) + Lat, so the simulated past is void from the flow's release on
 *                       (nothing is void if it has not been released yet, or if max(start, release) does not change):
 *                       the next run continues from the newest snapshot before that time.  A flow WITHOUT predecessors
 *                       sits in the sorted initial-activation lists: the tables are rebuilt and the next run starts at 0.
 *   phs_rollback        declares the simulated past void from time t_s on (results become unavailable until the next run).
 *   phs_gc              PAPER.md L130: drops the snapshots no rollback to a time >= t_s can need.
 * phs_add_flows / phs_add_collective* / phs_add_spans after phs_finalize are late submissions (L124): the tables are
 * rebuilt (the units may merge) and the next run starts at t = 0; results are those of a fresh run either way, the
 * simulation being deterministic -- the oracle (oracle/orc_netsim.c) rolls back exactly as the paper describes and
 * pins that equality. */
phs_status phs_set_snapshots(phs_sim *sim, int32_t n);
phs_status phs_update_flow_start(phs_sim *sim, int32_t instance, int64_t flow, double start_time_s);
phs_status phs_rollback(phs_sim *sim, double t_s);
phs_status phs_gc(phs_sim *sim, double t_s);

phs_status phs_num_flows(const phs_sim *sim, int32_t instance, int64_t *out);
phs_status phs_total_flows(const phs_sim *sim, int64_t *out);
phs_status phs_num_collectives(const phs_sim *sim, int32_t instance, int32_t *out);
/* out[n] with n == flows of the instance; out_is_device != 0: `out` is a device pointer filled on the run's stream. */
phs_status phs_get_completion_times(const phs_sim *sim, int32_t instance, double *out, int64_t n, int32_t out_is_device);
phs_status phs_get_bottlenecks(const phs_sim *sim, int32_t instance, int32_t *out, int64_t n, int32_t out_is_device);
/* All instances at once, concatenated in instance order: out[total_flows]. */
phs_status phs_get_all_completion_times(const phs_sim *sim, double *out, int64_t n, int32_t out_is_device);
phs_status phs_get_all_bottlenecks(const phs_sim *sim, int32_t *out, int64_t n, int32_t out_is_device);
/* Per-collective finish time = max completion time over its flows (computed on the GPU). */
phs_status phs_get_collective_times(const phs_sim *sim, int32_t instance, double *out, int32_t n);
phs_status phs_get_event_log(const phs_sim *sim, int32_t instance, phs_event *out, int64_t cap, int64_t *n_events);
/* Routing / decomposition artefacts (host side), for integer parity: paths as CSR off[F+1], links[cap];
 * preds as CSR. */
phs_status phs_num_path_entries(const phs_sim *sim, int32_t instance, int64_t *out);
phs_status phs_get_paths(const phs_sim *sim, int32_t instance, int64_t *off, int32_t *links, int64_t cap);
/* The transpose, link -> flow incidence (PAPER.md L98 routing): off[n_links + 1], flows[cap] with
 * cap >= phs_num_path_entries: per link the flows whose path crosses it, ascending flow id. */
phs_status phs_get_link_flows(const phs_sim *sim, int32_t instance, int64_t *off, int32_t *flows, int64_t cap);
phs_status phs_get_preds(const phs_sim *sim, int32_t instance, int64_t *off, int32_t *preds, int64_t cap,
                         int64_t *n_entries);
phs_status phs_get_flow_table(const phs_sim *sim, int32_t instance, int32_t *src, int32_t *dst, double *bytes,
                              double *latency_s, int64_t n);
phs_status phs_get_counters(const phs_sim *sim, phs_counters *out);
/* Name of the kernel path the last run used for the largest unit of `instance`: "cta", "cluster", "window", "grid". */
const char *phs_instance_path(const phs_sim *sim, int32_t instance);
const char *phs_last_error(void); /* thread-local; valid until the next call on this thread */

#ifdef __cplusplus
}
#endif
#endif
