// phs_api.cu -- the C-ABI of libphs (include/phs.h): handle, host-side submission calls and the result getters
// (a10).  Table construction, the batch scheduler and phs_run are in phs_schedule.cu.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <numeric>

#include "phs_sim.h"

using namespace phs;

namespace {
thread_local std::string g_err;
}  // namespace

phs_status phs_fail(phs_status code, const std::string &msg) {
  g_err = msg;
  return code;
}
#define fail phs_fail

extern "C" {

const char *phs_last_error(void) { return g_err.c_str(); }

phs_status phs_create_topology(const phs_topology_desc *desc, uint64_t seed, int32_t batch, phs_sim **out) {
  PHS_API_BEGIN
  if (!desc || !out) return fail(PHS_EINVAL, "null argument");
  if (batch <= 0) return fail(PHS_EINVAL, "batch must be positive");
  std::string why;
  phs_status st = Fabric::validate(*desc, &why);
  if (st != PHS_OK) return fail(st, why);
  std::unique_ptr<phs_sim> s(new phs_sim());  // bad_alloc -> PHS_ENOMEM (PHS_API_END)
  s->desc = *desc;
  s->seed = seed;
  s->batch = batch;
  s->fab.reset(new Fabric(*desc));
  s->inst.resize((size_t)batch);
  for (int32_t i = 0; i < batch; ++i) s->inst[i].seed = seed + (uint64_t)i;
  *out = s.release();
  return PHS_OK;
  PHS_API_END
}

phs_status phs_create_topology_graph(int32_t n_gpus, int32_t n_nodes, int32_t n_links, const int32_t *link_from,
                                     const int32_t *link_to, const double *cap_Bps, const double *latency_s,
                                     int32_t compute_lanes, uint64_t seed, int32_t batch, phs_sim **out) {
  PHS_API_BEGIN
  if (!out || !link_from || !link_to || !cap_Bps || !latency_s || n_links < 1) return fail(PHS_EINVAL, "null argument");
  if (batch <= 0) return fail(PHS_EINVAL, "batch must be positive");
  GraphLinks g;
  g.n_gpus = n_gpus;
  g.n_nodes = n_nodes;
  g.compute_lanes = compute_lanes;
  g.from.assign(link_from, link_from + n_links);
  g.to.assign(link_to, link_to + n_links);
  g.cap.assign(cap_Bps, cap_Bps + n_links);
  g.lat.assign(latency_s, latency_s + n_links);
  std::string why;
  phs_status st = Fabric::validate_graph(g, &why);
  if (st != PHS_OK) return fail(st, why);
  std::unique_ptr<phs_sim> s(new phs_sim());
  s->desc = phs_topology_desc{};
  s->desc.kind = 3;
  s->desc.n_hosts = n_gpus;
  s->desc.gpus_per_host = 1;
  s->desc.compute_lanes = compute_lanes;
  s->seed = seed;
  s->batch = batch;
  s->fab.reset(new Fabric(std::move(g)));
  s->inst.resize((size_t)batch);
  for (int32_t i = 0; i < batch; ++i) s->inst[i].seed = seed + (uint64_t)i;
  *out = s.release();
  return PHS_OK;
  PHS_API_END
}

void phs_destroy(phs_sim *sim) { delete sim; }

phs_status phs_num_links(const phs_sim *sim, int32_t *out) {
  PHS_API_BEGIN
  if (!sim || !out) return fail(PHS_EINVAL, "null argument");
  *out = sim->fab->n_links();
  return PHS_OK;
  PHS_API_END
}

phs_status phs_batch(const phs_sim *sim, int32_t *out) {
  PHS_API_BEGIN
  if (!sim || !out) return fail(PHS_EINVAL, "null argument");
  *out = sim->batch;
  return PHS_OK;
  PHS_API_END
}

// The instance with every submitted collective expanded into flows.  Expansion is deferred bookkeeping, not a change
// of the handle's observable state, hence the const_cast.
static const Instance &expanded(const phs_sim *sim, int32_t instance) {
  Instance &in = const_cast<phs_sim *>(sim)->inst[(size_t)instance];
  expand_pending(*sim->fab, in);
  return in;
}

static phs_status check_instance(const phs_sim *sim, int32_t instance, bool allow_all) {
  if (!sim) return fail(PHS_EINVAL, "null handle");
  if (instance == -1 && allow_all) return PHS_OK;
  if (instance < 0 || instance >= sim->batch) return fail(PHS_EINVAL, "instance out of range");
  return PHS_OK;
}

// multi-device handle after phs_finalize: the shard that holds `instance` (nullptr otherwise), the instance's index
// there and the shard's device
static phs_sim *shard_of(const phs_sim *sim, int32_t instance, int32_t *local, int *dev) {
  if (!sim || sim->shards.empty() || instance < 0 || instance >= sim->batch) return nullptr;
  const size_t k = (size_t)(std::upper_bound(sim->shard_first.begin(), sim->shard_first.end(), instance) -
                            sim->shard_first.begin()) - 1;
  *local = instance - sim->shard_first[k];
  *dev = sim->devices[k];
  return sim->shards[k].get();
}

phs_status phs_set_devices(phs_sim *sim, int32_t n, const int32_t *device_ids) {
  PHS_API_BEGIN
  if (!sim || n < 1 || !device_ids) return fail(PHS_EINVAL, "bad device list");
  if (sim->finalized) return fail(PHS_ESTATE, "the devices must be chosen before phs_finalize");
  for (int i = 0; i < n; ++i)
    if (device_ids[i] < 0) return fail(PHS_EINVAL, "negative device id");
  if (n > sim->batch) return fail(PHS_EINVAL, "more devices than instances: a single instance does not shard");
  sim->devices.assign(device_ids, device_ids + n);
  return PHS_OK;
  PHS_API_END
}

phs_status phs_instance_device(const phs_sim *sim, int32_t instance, int32_t *out) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  if (!out) return fail(PHS_EINVAL, "null output");
  int32_t li = 0;
  int dev = 0;
  if (shard_of(sim, instance, &li, &dev)) {
    *out = dev;
    return PHS_OK;
  }
  PHS_CUDA(cudaGetDevice(&dev));
  *out = sim->devices.size() == 1 ? sim->devices[0] : dev;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_set_link_capacities(phs_sim *sim, int32_t instance, const double *cap) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, true);
  if (st != PHS_OK) return st;
  if (!cap) return fail(PHS_EINVAL, "null capacities");
  if (sim->finalized) return fail(PHS_ESTATE, "instance set is frozen after phs_finalize");
  const int L = sim->fab->n_links();
  for (int l = 0; l < L; ++l)
    if (!(cap[l] > 0.0) || !(cap[l] < 0x1p42)) return fail(PHS_EINVAL, "capacity must be in (0, 2^42) byte/s");
  const int lo = instance < 0 ? 0 : instance, hi = instance < 0 ? sim->batch : instance + 1;
  for (int i = lo; i < hi; ++i) sim->inst[i].cap.assign(cap, cap + L);
  return PHS_OK;
  PHS_API_END
}

phs_status phs_set_link_capacities_batch(phs_sim *sim, const double *cap) {
  PHS_API_BEGIN
  if (!sim || !cap) return fail(PHS_EINVAL, "null argument");
  if (sim->finalized) return fail(PHS_ESTATE, "instance set is frozen after phs_finalize");
  const size_t L = (size_t)sim->fab->n_links(), n = L * (size_t)sim->batch;
  for (size_t k = 0; k < n; ++k)  // validate everything first so that a failure changes nothing
    if (!(cap[k] > 0.0) || !(cap[k] < 0x1p42)) return fail(PHS_EINVAL, "capacity must be in (0, 2^42) byte/s");
  for (int i = 0; i < sim->batch; ++i) sim->inst[i].cap.assign(cap + (size_t)i * L, cap + (size_t)(i + 1) * L);
  return PHS_OK;
  PHS_API_END
}

phs_status phs_get_link_capacities(const phs_sim *sim, int32_t instance, double *cap) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  if (!cap) return fail(PHS_EINVAL, "null output");
  const int L = sim->fab->n_links();
  const Instance &in = sim->inst[instance];
  for (int l = 0; l < L; ++l) cap[l] = in.cap.empty() ? sim->fab->default_capacity(l) : in.cap[l];
  return PHS_OK;
  PHS_API_END
}

phs_status phs_add_collective(phs_sim *sim, int32_t instance, int32_t kind, const int32_t *ranks, int32_t n_ranks,
                              double bytes, double start, const int32_t *after, int32_t n_after, int32_t *out_id) {
  return phs_add_collective_ex(sim, instance, kind, ranks, n_ranks, bytes, start, after, n_after, 1, out_id);
}

phs_status phs_add_collective_ex(phs_sim *sim, int32_t instance, int32_t kind, const int32_t *ranks, int32_t n_ranks,
                                 double bytes, double start, const int32_t *after, int32_t n_after, int32_t chunks,
                                 int32_t *out_id) {
  return phs_add_collective_full(sim, instance, kind, ranks, n_ranks, bytes, start, after, n_after, nullptr, 0, chunks,
                                 out_id);
}

phs_status phs_add_spans(phs_sim *sim, int32_t instance, int64_t n, const int32_t *gpu, const int32_t *lane,
                         const double *duration, const double *start, const int64_t *dep_off, const int64_t *dep_ids,
                         int64_t *out_first) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, true);
  if (st != PHS_OK) return st;
  if (sim->finalized && !sim->shards.empty()) return fail(PHS_ESTATE, "late submissions are not supported on a multi-device handle");
  if (sim->finalized) phs_unfinalize(sim);  // a late submission: the tables are rebuilt by the next run
  const int lo = instance < 0 ? 0 : instance, hi = instance < 0 ? sim->batch : instance + 1;
  if (instance < 0)
    for (int i = 1; i < sim->batch; ++i)
      if (sim->inst[i].n_flows() != sim->inst[0].n_flows())
        return fail(PHS_ESTATE, "instance -1 needs the same number of flows in every instance");
  const int64_t first = sim->inst[lo].n_flows();
  std::string why;
  for (int i = lo; i < hi; ++i) {
    st = append_spans(*sim->fab, sim->inst[i], n, gpu, lane, duration, start, dep_off, dep_ids, &why);
    if (st != PHS_OK) return fail(st, why);
  }
  if (out_first) *out_first = first;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_add_collective_full(phs_sim *sim, int32_t instance, int32_t kind, const int32_t *ranks, int32_t n_ranks,
                                   double bytes, double start, const int32_t *after, int32_t n_after,
                                   const int64_t *after_flows, int32_t n_after_flows, int32_t chunks, int32_t *out_id) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, true);
  if (st != PHS_OK) return st;
  if (sim->finalized && !sim->shards.empty()) return fail(PHS_ESTATE, "late submissions are not supported on a multi-device handle");
  if (sim->finalized) phs_unfinalize(sim);  // a late submission: the tables are rebuilt by the next run
  const int lo = instance < 0 ? 0 : instance, hi = instance < 0 ? sim->batch : instance + 1;
  if (instance < 0)
    for (int i = 1; i < sim->batch; ++i)
      if (sim->inst[i].colls.size() != sim->inst[0].colls.size())
        return fail(PHS_ESTATE, "instance -1 needs the same number of collectives in every instance");
  std::string why;
  for (int i = lo; i < hi; ++i) {
    st = append_collective(*sim->fab, sim->inst[i], kind, ranks, n_ranks, bytes, start, after, n_after, after_flows,
                           n_after_flows, chunks, &why);
    if (st != PHS_OK) return fail(st, why);  // validation fails on the first instance, before any mutation
  }
  if (out_id) *out_id = (int32_t)sim->inst[lo].colls.size() - 1;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_add_collective_batch(phs_sim *sim, int32_t kind, const int32_t *ranks, int32_t n_ranks,
                                    const double *bytes, const double *start, const int32_t *after, int32_t n_after,
                                    int32_t *out_id) {
  PHS_API_BEGIN
  if (!sim || !bytes) return fail(PHS_EINVAL, "null argument");
  if (sim->finalized && !sim->shards.empty()) return fail(PHS_ESTATE, "late submissions are not supported on a multi-device handle");
  if (sim->finalized) phs_unfinalize(sim);  // a late submission: the tables are rebuilt by the next run
  for (int i = 1; i < sim->batch; ++i)
    if (sim->inst[i].colls.size() != sim->inst[0].colls.size())
      return fail(PHS_ESTATE, "batch add needs the same number of collectives in every instance");
  for (int i = 0; i < sim->batch; ++i) {  // validate all sizes first so that a failure leaves nothing half-added
    if (!(bytes[i] > 0.0) || !std::isfinite(bytes[i])) return fail(PHS_EINVAL, "bytes must be positive and finite");
    if (start && (!(start[i] >= 0.0) || !std::isfinite(start[i]))) return fail(PHS_EINVAL, "bad start_time_s");
  }
  // the arguments shared by all instances (kind, ranks, after) fail on instance 0, before anything is added.  Only
  // the descriptor is recorded here: the flows are expanded per instance on the host threads of phs_finalize.
  std::string why;
  phs_status st0 = append_collective(*sim->fab, sim->inst[0], kind, ranks, n_ranks, bytes[0], start ? start[0] : 0.0, after,
                                     n_after, nullptr, 0, 1, &why);
  if (st0 != PHS_OK) return fail(st0, why);
  // the other instances record the same descriptor with their own size and start time; what depends on the instance
  // (its flow count so far: the 2^31 limit) is still checked
  for (int i = 1; i < sim->batch; ++i) {
    phs_status sti = append_collective(*sim->fab, sim->inst[i], kind, ranks, n_ranks, bytes[i], start ? start[i] : 0.0,
                                       after, n_after, nullptr, 0, 1, &why, true);
    if (sti != PHS_OK) return fail(sti, why);
  }
  if (out_id) *out_id = (int32_t)sim->inst[0].colls.size() - 1;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_add_flows(phs_sim *sim, int32_t instance, int64_t n, const int32_t *src, const int32_t *dst,
                         const double *bytes, const double *start, const int64_t *dep_off, const int64_t *dep_ids,
                         const int32_t *conn_id, int64_t *out_first) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, true);
  if (st != PHS_OK) return st;
  if (sim->finalized && !sim->shards.empty()) return fail(PHS_ESTATE, "late submissions are not supported on a multi-device handle");
  if (sim->finalized) phs_unfinalize(sim);  // a late submission: the tables are rebuilt by the next run
  const int lo = instance < 0 ? 0 : instance, hi = instance < 0 ? sim->batch : instance + 1;
  if (instance < 0)
    for (int i = 1; i < sim->batch; ++i)
      if (sim->inst[i].n_flows() != sim->inst[0].n_flows())
        return fail(PHS_ESTATE, "instance -1 needs the same number of flows in every instance");
  const int64_t first = sim->inst[lo].n_flows();
  std::string why;
  for (int i = lo; i < hi; ++i) {
    st = append_flows(*sim->fab, sim->inst[i], n, src, dst, bytes, start, dep_off, dep_ids, conn_id, &why);
    if (st != PHS_OK) return fail(st, why);
  }
  if (out_first) *out_first = first;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_enable_event_log(phs_sim *sim, int32_t enable) {
  PHS_API_BEGIN
  if (!sim) return fail(PHS_EINVAL, "null handle");
  if (sim->finalized) return fail(PHS_ESTATE, "event log must be chosen before phs_finalize");
  sim->want_log = enable != 0;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_set_scheduler(phs_sim *sim, int32_t path, int32_t cta_slots) {
  PHS_API_BEGIN
  if (!sim) return fail(PHS_EINVAL, "null handle");
  if (path < 0 || path > 4 || cta_slots < 0) return fail(PHS_EINVAL, "bad scheduler policy");
  if (sim->finalized) return fail(PHS_ESTATE, "scheduler policy must be chosen before phs_finalize");
  sim->policy_path = path;
  sim->policy_slots = cta_slots;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_enable_history(phs_sim *sim, int64_t max_records) {
  PHS_API_BEGIN
  if (!sim) return fail(PHS_EINVAL, "null handle");
  if (max_records < 0) return fail(PHS_EINVAL, "max_records must be >= 0");
  if (sim->finalized) return fail(PHS_ESTATE, "history must be chosen before phs_finalize");
  sim->hist_cap = max_records;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_set_decomposition(phs_sim *sim, int32_t enable) {
  PHS_API_BEGIN
  if (!sim) return fail(PHS_EINVAL, "null handle");
  if (sim->finalized) return fail(PHS_ESTATE, "decomposition must be chosen before phs_finalize");
  sim->decompose = enable != 0;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_set_windows(phs_sim *sim, int32_t enable) {
  PHS_API_BEGIN
  if (!sim) return fail(PHS_EINVAL, "null handle");
  if (sim->finalized) return fail(PHS_ESTATE, "the window schedule must be chosen before phs_finalize");
  sim->windows = enable != 0;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_num_flows(const phs_sim *sim, int32_t instance, int64_t *out) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  if (!out) return fail(PHS_EINVAL, "null output");
  *out = sim->inst[instance].n_flows();
  return PHS_OK;
  PHS_API_END
}

phs_status phs_total_flows(const phs_sim *sim, int64_t *out) {
  PHS_API_BEGIN
  if (!sim || !out) return fail(PHS_EINVAL, "null argument");
  int64_t t = 0;
  for (const Instance &in : sim->inst) t += in.n_flows();
  *out = t;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_num_collectives(const phs_sim *sim, int32_t instance, int32_t *out) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  if (!out) return fail(PHS_EINVAL, "null output");
  *out = (int32_t)sim->inst[instance].colls.size();
  return PHS_OK;
  PHS_API_END
}

phs_status phs_num_path_entries(const phs_sim *sim, int32_t instance, int64_t *out) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  if (!out) return fail(PHS_EINVAL, "null output");
  *out = (int64_t)expanded(sim, instance).path.size();
  return PHS_OK;
  PHS_API_END
}

phs_status phs_get_paths(const phs_sim *sim, int32_t instance, int64_t *off, int32_t *links, int64_t cap) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  const Instance &in = expanded(sim, instance);
  if (!off || !links || cap < (int64_t)in.path.size()) return fail(PHS_EINVAL, "output too small");
  for (size_t f = 0; f < in.path_off.size(); ++f) off[f] = in.path_off[f];
  std::copy(in.path.begin(), in.path.end(), links);
  return PHS_OK;
  PHS_API_END
}

// a3: the transpose of the flow -> link incidence (lf_off[n_links + 1], lf[sum of path lengths]):
// per link the flows that cross it, ascending flow id.  Counting sort over the path entries.
phs_status phs_get_link_flows(const phs_sim *sim, int32_t instance, int64_t *off, int32_t *flows, int64_t cap) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  const Instance &in = expanded(sim, instance);
  if (!off || !flows || cap < (int64_t)in.path.size()) return fail(PHS_EINVAL, "output too small");
  const int32_t L = sim->fab->n_links();
  std::fill(off, off + L + 1, (int64_t)0);
  for (int32_t l : in.path) off[l + 1]++;
  for (int32_t l = 0; l < L; ++l) off[l + 1] += off[l];
  std::vector<int64_t> cur(off, off + L);
  for (size_t f = 0; f + 1 < in.path_off.size(); ++f)
    for (uint32_t e = in.path_off[f]; e < in.path_off[f + 1]; ++e) flows[cur[(size_t)in.path[e]]++] = (int32_t)f;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_get_preds(const phs_sim *sim, int32_t instance, int64_t *off, int32_t *preds, int64_t cap,
                         int64_t *n_entries) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  const Instance &in = expanded(sim, instance);
  if (!n_entries) return fail(PHS_EINVAL, "null n_entries");
  *n_entries = (int64_t)in.pred.size();
  if (off)
    for (size_t f = 0; f < in.pred_off.size(); ++f) off[f] = in.pred_off[f];
  if (preds) {
    if (cap < (int64_t)in.pred.size()) return fail(PHS_EINVAL, "output too small");
    std::copy(in.pred.begin(), in.pred.end(), preds);
  }
  return PHS_OK;
  PHS_API_END
}

phs_status phs_get_flow_table(const phs_sim *sim, int32_t instance, int32_t *src, int32_t *dst, double *bytes,
                              double *lat, int64_t n) {
  PHS_API_BEGIN
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  const Instance &in = expanded(sim, instance);
  if (n != in.n_flows()) return fail(PHS_EINVAL, "n must equal the instance's flow count");
  if (src) std::copy(in.src.begin(), in.src.end(), src);
  if (dst) std::copy(in.dst.begin(), in.dst.end(), dst);
  if (bytes) std::copy(in.bytes.begin(), in.bytes.end(), bytes);
  if (lat) std::copy(in.lat.begin(), in.lat.end(), lat);
  return PHS_OK;
  PHS_API_END
}

}  // extern "C"

// ================================================================================================ results (a10)
namespace {
template <typename T>
phs_status fetch(const phs_sim *sim, const T *dev, int64_t first, int64_t count, T *out, int32_t out_is_device) {
  if (count == 0) return PHS_OK;
  std::unique_ptr<DeviceGuard> on_device;  // phs_set_devices with one device
  if (sim->devices.size() == 1) on_device.reset(new DeviceGuard(sim->devices[0]));
  const size_t bytes = sizeof(T) * (size_t)count;
  if (!out_is_device && bytes >= (256u << 10)) {
    // host output: through the page-locked staging area (phs_finalize sized it for the tables, so results fit),
    // then into the caller's pageable buffer with host threads -- several times faster than a pageable D2H copy
    StagingArea &stage = staging_area();
    std::lock_guard<std::mutex> lock(stage.mu);
    if (stage.pinned && stage.cap >= bytes) {
      PHS_CUDA(cudaMemcpyAsync(stage.p, dev + first, bytes, cudaMemcpyDeviceToHost, sim->last_stream));
      PHS_CUDA(cudaStreamSynchronize(sim->last_stream));
      const size_t piece = 4u << 20;
      const int n_pieces = (int)((bytes + piece - 1) / piece);
      parallel_for(n_pieces, [&](int k) {
        const size_t lo = (size_t)k * piece, len = std::min(piece, bytes - lo);
        std::memcpy((unsigned char *)out + lo, stage.p + lo, len);
      });
      return PHS_OK;
    }
  }
  PHS_CUDA(cudaMemcpyAsync(out, dev + first, bytes, out_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost,
                           sim->last_stream));
  if (!out_is_device) PHS_CUDA(cudaStreamSynchronize(sim->last_stream));
  return PHS_OK;
}
}  // namespace

extern "C" {

phs_status phs_get_completion_times(const phs_sim *sim, int32_t instance, double *out, int64_t n, int32_t dev) {
  PHS_API_BEGIN
  {
    int32_t li_ = 0;
    int dev_ = 0;
    if (phs_sim *sh_ = shard_of(sim, instance, &li_, &dev_)) {
      DeviceGuard guard_(dev_);
      return phs_get_completion_times(sh_, li_, out, n, dev);
    }
  }
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  if (!sim->ran) return fail(PHS_ESTATE, "phs_run has not completed");
  if (!out || n != sim->inst[instance].n_flows()) return fail(PHS_EINVAL, "n must equal the instance's flow count");
  return fetch(sim, sim->d_tdone.p, sim->flow_base[instance], n, out, dev);
  PHS_API_END
}

phs_status phs_get_bottlenecks(const phs_sim *sim, int32_t instance, int32_t *out, int64_t n, int32_t dev) {
  PHS_API_BEGIN
  {
    int32_t li_ = 0;
    int dev_ = 0;
    if (phs_sim *sh_ = shard_of(sim, instance, &li_, &dev_)) {
      DeviceGuard guard_(dev_);
      return phs_get_bottlenecks(sh_, li_, out, n, dev);
    }
  }
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  if (!sim->ran) return fail(PHS_ESTATE, "phs_run has not completed");
  if (!out || n != sim->inst[instance].n_flows()) return fail(PHS_EINVAL, "n must equal the instance's flow count");
  return fetch(sim, sim->d_bneck.p, sim->flow_base[instance], n, out, dev);
  PHS_API_END
}

phs_status phs_get_all_completion_times(const phs_sim *sim, double *out, int64_t n, int32_t dev) {
  PHS_API_BEGIN
  if (!sim || !out) return fail(PHS_EINVAL, "null argument");
  if (!sim->shards.empty()) {  // one block per device, concatenated in instance order
    if (dev) return fail(PHS_EINVAL, "a multi-device handle returns host arrays only");
    if (n != sim->total_flows) return fail(PHS_EINVAL, "n must equal the total flow count");
    for (size_t k = 0; k < sim->shards.size(); ++k) {
      DeviceGuard guard_(sim->devices[k]);
      const phs_sim *sh = sim->shards[k].get();
      phs_status st = phs_get_all_completion_times(sh, out + sim->flow_base[(size_t)sim->shard_first[k]], sh->total_flows, 0);
      if (st != PHS_OK) return st;
    }
    return PHS_OK;
  }
  if (!sim->ran) return fail(PHS_ESTATE, "phs_run has not completed");
  if (n != sim->total_flows) return fail(PHS_EINVAL, "n must equal the total flow count");
  return fetch(sim, sim->d_tdone.p, 0, n, out, dev);
  PHS_API_END
}

phs_status phs_get_all_bottlenecks(const phs_sim *sim, int32_t *out, int64_t n, int32_t dev) {
  PHS_API_BEGIN
  if (!sim || !out) return fail(PHS_EINVAL, "null argument");
  if (!sim->shards.empty()) {
    if (dev) return fail(PHS_EINVAL, "a multi-device handle returns host arrays only");
    if (n != sim->total_flows) return fail(PHS_EINVAL, "n must equal the total flow count");
    for (size_t k = 0; k < sim->shards.size(); ++k) {
      DeviceGuard guard_(sim->devices[k]);
      const phs_sim *sh = sim->shards[k].get();
      phs_status st = phs_get_all_bottlenecks(sh, out + sim->flow_base[(size_t)sim->shard_first[k]], sh->total_flows, 0);
      if (st != PHS_OK) return st;
    }
    return PHS_OK;
  }
  if (!sim->ran) return fail(PHS_ESTATE, "phs_run has not completed");
  if (n != sim->total_flows) return fail(PHS_EINVAL, "n must equal the total flow count");
  return fetch(sim, sim->d_bneck.p, 0, n, out, dev);
  PHS_API_END
}

phs_status phs_get_collective_times(const phs_sim *sim, int32_t instance, double *out, int32_t n) {
  PHS_API_BEGIN
  {
    int32_t li_ = 0;
    int dev_ = 0;
    if (phs_sim *sh_ = shard_of(sim, instance, &li_, &dev_)) {
      DeviceGuard guard_(dev_);
      return phs_get_collective_times(sh_, li_, out, n);
    }
  }
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  if (!sim->ran) return fail(PHS_ESTATE, "phs_run has not completed");
  if (!out || n != (int32_t)sim->inst[instance].colls.size()) return fail(PHS_EINVAL, "n must equal the collective count");
  return fetch(sim, sim->d_coll_t.p, sim->coll_base[instance], (int64_t)n, out, 0);
  PHS_API_END
}

phs_status phs_get_event_log(const phs_sim *sim, int32_t instance, phs_event *out, int64_t cap, int64_t *n_events) {
  PHS_API_BEGIN
  {
    int32_t li_ = 0;
    int dev_ = 0;
    if (phs_sim *sh_ = shard_of(sim, instance, &li_, &dev_)) {
      DeviceGuard guard_(dev_);
      return phs_get_event_log(sh_, li_, out, cap, n_events);
    }
  }
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  if (!sim->ran) return fail(PHS_ESTATE, "phs_run has not completed");
  if (!sim->want_log) return fail(PHS_ESTATE, "event log was not enabled");
  if (!n_events) return fail(PHS_EINVAL, "null n_events");
  *n_events = sim->h_res[sim->unit_first[instance]].n_events;  // with the log on, an instance is one unit
  if (!out) return PHS_OK;
  return fetch(sim, sim->d_log.p, sim->h_desc[sim->unit_first[instance]].log_base, std::min<int64_t>(cap, *n_events),
               out, 0);
  PHS_API_END
}

phs_status phs_get_flow_history(const phs_sim *sim, int32_t instance, int64_t *off, double *t, double *rate,
                                int64_t cap, int64_t *n_records) {
  PHS_API_BEGIN
  {
    int32_t li_ = 0;
    int dev_ = 0;
    if (phs_sim *sh_ = shard_of(sim, instance, &li_, &dev_)) {
      DeviceGuard guard_(dev_);
      return phs_get_flow_history(sh_, li_, off, t, rate, cap, n_records);
    }
  }
  phs_status st = check_instance(sim, instance, false);
  if (st != PHS_OK) return st;
  if (!sim->ran) return fail(PHS_ESTATE, "phs_run has not completed");
  if (sim->hist_cap <= 0) return fail(PHS_ESTATE, "throughput history was not enabled");
  const uint32_t lo = (uint32_t)sim->flow_base[instance], hi = (uint32_t)sim->flow_base[instance + 1];
  auto by_flow = [](const HistRec &r, uint32_t f) { return r.flow < f; };
  const auto b = std::lower_bound(sim->h_hist.begin(), sim->h_hist.end(), lo, by_flow);
  const auto e = std::lower_bound(sim->h_hist.begin(), sim->h_hist.end(), hi, by_flow);
  const int64_t n = (int64_t)(e - b);
  if (n_records) *n_records = n;
  if (!t && !rate && !off) return PHS_OK;
  if (!t || !rate || !off || cap < n) return fail(PHS_EINVAL, "output too small");
  int64_t k = 0;
  auto it = b;
  for (uint32_t f = lo; f < hi; ++f) {
    off[f - lo] = k;
    for (; it != e && it->flow == f; ++it, ++k) {
      t[k] = it->t;
      rate[k] = it->rate;
    }
  }
  off[hi - lo] = k;
  return PHS_OK;
  PHS_API_END
}

phs_status phs_get_counters(const phs_sim *sim, phs_counters *out) {
  PHS_API_BEGIN
  if (!sim || !out) return fail(PHS_EINVAL, "null argument");
  if (!sim->ran) return fail(PHS_ESTATE, "phs_run has not completed");
  phs_counters c{};
  if (!sim->shards.empty()) {  // sums over the devices; kernel time = the slowest device (they run at once)
    for (const auto &sh : sim->shards) {
      phs_counters k{};
      phs_status st = phs_get_counters(sh.get(), &k);
      if (st != PHS_OK) return st;
      c.n_events += k.n_events; c.n_flow_events += k.n_flow_events; c.sum_active += k.sum_active;
      c.sum_par_rounds += k.sum_par_rounds; c.n_kernel_launches += k.n_kernel_launches; c.h2d_bytes += k.h2d_bytes;
      c.n_windows += k.n_windows; c.resumed_units += k.resumed_units;
      c.max_active = std::max(c.max_active, k.max_active); c.max_slots = std::max(c.max_slots, k.max_slots);
      c.cluster_size = std::max(c.cluster_size, k.cluster_size);
      c.clusters_resident = std::max(c.clusters_resident, k.clusters_resident);
      c.window_gang = std::max(c.window_gang, k.window_gang); c.grid_ctas = std::max(c.grid_ctas, k.grid_ctas);
      c.main_kernel_ms = std::max(c.main_kernel_ms, k.main_kernel_ms);
      c.resumed_from_s = k.resumed_from_s;
    }
    *out = c;
    return PHS_OK;
  }
  for (size_t i = 0; i < sim->units.size(); ++i) {
    c.n_events += sim->h_res[i].n_events;
    c.sum_active += sim->h_res[i].sum_active;
    c.sum_par_rounds += sim->h_res[i].sum_par_rounds;
    c.max_active = std::max(c.max_active, sim->h_res[i].max_active);
    c.max_slots = std::max(c.max_slots, sim->h_res[i].max_slots);
    c.n_windows += sim->h_res[i].n_windows;
  }
  c.cluster_size = sim->scratch_cs;
  c.window_gang = sim->win_gang_used;
  c.grid_ctas = sim->grid_ctas;
  c.clusters_resident = sim->clusters_resident;
  c.resumed_units = sim->resumed_units;
  c.n_flow_events = 2 * sim->total_flows;
  c.n_kernel_launches = sim->n_launches;
  c.h2d_bytes = sim->h2d_bytes;
  c.main_kernel_ms = sim->main_kernel_ms;
  c.resumed_from_s = sim->resumed_from;
  *out = c;
  return PHS_OK;
  PHS_API_END
}

const char *phs_instance_path(const phs_sim *sim, int32_t instance) {
  if (!sim || instance < 0 || instance >= sim->batch || !sim->ran) return "";
  {
    int32_t li_ = 0;
    int dev_ = 0;
    if (phs_sim *sh_ = shard_of(sim, instance, &li_, &dev_)) return phs_instance_path(sh_, li_);
  }
  int best = sim->unit_first[instance];  // the path of the instance's largest unit
  for (int u = best; u < sim->unit_first[instance + 1]; ++u)
    if (sim->units[u].n_flows > sim->units[best].n_flows) best = u;
  static const char *names[] = {"cta", "cluster", "window", "grid"};
  const int pth = sim->h_res[best].path;
  return pth >= 0 && pth < 4 ? names[pth] : "";
}

}  // extern "C"
