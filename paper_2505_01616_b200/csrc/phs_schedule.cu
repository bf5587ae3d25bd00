// phs_schedule.cu -- phs_finalize (simulation units, device-resident tables, static part of the batch scheduler)
// and phs_run (launches, overflow handling, throughput-history fetch): SURVEY.md 8(a) a9.  No CPU fallback
// exists: without a usable CUDA device both fail with PHS_ECUDA.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <numeric>
#include <type_traits>

#include "phs_sim.h"
#include <chrono>
#include <cstdio>
#include <cstdlib>

using namespace phs;

namespace phs {
StagingArea &staging_area() {
  static StagingArea area;  // never freed: the CUDA context may be gone when static destructors run
  return area;
}
}  // namespace phs

#define fail phs_fail
#define PHS_DBG(...) do { if (getenv("PHS_DEBUG")) { fprintf(stderr, "[phs dbg] " __VA_ARGS__); fputc('\n', stderr); fflush(stderr); } } while (0)

// ================================================================================================ window path plan
namespace {

// Decides whether unit `u` runs on the window path and with how many CTAs (a9), for slot estimates scaled by
// `scale` quarters, and writes the ownership tables of its gang: the unit's static link components are dealt to the
// CTAs largest first, each to the CTA with the fewest flows so far; links and components get indices local to their
// owner.  A unit that does not go there keeps the identity tables (owner 0).
bool plan_window_unit(phs_sim *sim, int u, size_t smem_max, int64_t scale) {
  phs_sim::Unit &un = sim->units[(size_t)u];
  const int32_t *lcomp = sim->h_lcomp.data() + un.link_base;
  uint32_t *lloc = sim->h_lloc.data() + un.link_base, *cown = sim->h_cown.data() + un.comp_base;
  const int32_t *cflows = sim->comp_flows.data() + un.comp_base, *clinks = sim->comp_links.data() + un.comp_base;
  un.win_gang = 0;
  for (int l = 0; l < un.n_links; ++l) lloc[l] = (uint32_t)l;
  for (int c = 0; c < un.n_comps; ++c) cown[c] = (uint32_t)c;
  double threshold = 4.0;  // estimated flow events per window from which the window schedule pays (measured: cfg1, with
                           // 0.4, is faster one event at a time; cfg2, with ~100, is 30 x faster in windows)
  if (const char *ev = getenv("PHS_WIN_DENSITY")) threshold = atof(ev);
  const bool forced = sim->policy_path == 3;  // phs_set_scheduler: every eligible unit, whatever its density
  if (!sim->windows || sim->want_log || sim->hist_cap > 0 || (sim->policy_path != 0 && !forced) || un.n_flows == 0)
    return false;
  // small units stay on the CTA path: many of them are resident per SM there, and a batch of them is bound by
  // instruction throughput, not by the length of one unit's event chain
  if (!(sim->h_desc[(size_t)u].lmin > 0.0) || (!forced && (!(un.density >= threshold) || un.n_flows < 8192))) return false;
  // gang size: about 16 components per CTA (measured on cfg2's 128-component unit: 8 and 16 CTAs tie, 4 are a third
  // slower), more if the unit does not fit otherwise
  int want_gang = 1;
  while (want_gang < 16 && un.n_comps > 16 * want_gang) want_gang *= 2;
  const int min_gang = forced ? std::max(1, sim->policy_slots) : want_gang;
  std::vector<int32_t> by_size((size_t)un.n_comps);
  std::iota(by_size.begin(), by_size.end(), 0);
  std::stable_sort(by_size.begin(), by_size.end(), [&](int a, int b) { return cflows[a] > cflows[b]; });
  for (int K = 1; K <= 16; K *= 2) {
    if (K < min_gang && un.n_comps >= K * 2) continue;
    if (K > 1 && un.n_comps < (forced ? K : 2 * K)) break;  // a gang needs components to share out
    std::vector<int64_t> kflows((size_t)K, 0);
    std::vector<int32_t> klinks((size_t)K, 0), kcomps((size_t)K, 0), owner((size_t)un.n_comps, 0);
    for (int c : by_size) {
      const int k = (int)(std::min_element(kflows.begin(), kflows.end()) - kflows.begin());
      owner[(size_t)c] = k;
      kflows[(size_t)k] += cflows[c];
      klinks[(size_t)k] += clinks[c];
      kcomps[(size_t)k]++;
    }
    const int Lm = *std::max_element(klinks.begin(), klinks.end());
    const int NCm = *std::max_element(kcomps.begin(), kcomps.end());
    const int64_t fmax = *std::max_element(kflows.begin(), kflows.end());
    if (Lm >= 65535) continue;
    // slots of the busiest CTA: its share of the unit's bound on PENDING + ACTIVE flows, a quarter on top
    int64_t slots = (int64_t)std::ceil((double)std::max<int64_t>(un.bound_cta, 32) * (double)fmax /
                                       (double)un.n_flows * 1.25 * (double)scale / 4.0) + 64;
    slots = std::min<int64_t>(slots, fmax + 32);
    slots = (slots + 31) / 32 * 32;
    if (window_smem_bytes(std::max(Lm, 1), std::max(NCm, 1), (int)slots) + 512 > smem_max) continue;
    std::vector<int32_t> next_link((size_t)K, 0), next_comp((size_t)K, 0);
    for (int c = 0; c < un.n_comps; ++c) cown[c] = ((uint32_t)owner[(size_t)c] << 24) | (uint32_t)next_comp[(size_t)owner[(size_t)c]]++;
    for (int l = 0; l < un.n_links; ++l) {
      const int k = owner[(size_t)lcomp[l]];
      lloc[l] = ((uint32_t)k << 24) | (uint32_t)next_link[(size_t)k]++;
    }
    un.win_gang = K;
    un.win_links = std::max(Lm, 1);
    un.win_comps = std::max(NCm, 1);
    un.win_slots = (int)slots;
    return true;
  }
  return false;
}

}  // namespace


// ================================================================================================ multi-GPU shards
namespace {

// fn(k, shard) on one host thread per shard, the shard's device current; returns the first error (message included)
template <typename Fn>
phs_status for_each_shard(phs_sim *sim, Fn fn) {
  const size_t n = sim->shards.size();
  std::vector<phs_status> rc(n, PHS_OK);
  std::vector<std::string> msg(n);
  std::vector<std::thread> pool;
  for (size_t k = 0; k < n; ++k)
    pool.emplace_back([&, k] {
      DeviceGuard guard(sim->devices[k]);
      rc[k] = fn(k, sim->shards[k].get());
      if (rc[k] != PHS_OK) msg[k] = phs_last_error();  // the message is thread-local: take it along
    });
  for (std::thread &th : pool) th.join();
  for (size_t k = 0; k < n; ++k)
    if (rc[k] != PHS_OK) return fail(rc[k], "device " + std::to_string(sim->devices[k]) + ": " + msg[k]);
  return PHS_OK;
}

// phs_set_devices with several devices: contiguous blocks of instances, one child handle per device
phs_status finalize_sharded(phs_sim *sim) {
  const int n = (int)sim->devices.size(), B = sim->batch;
  sim->flow_base.assign((size_t)B + 1, 0);
  sim->coll_base.assign((size_t)B + 1, 0);
  for (int i = 0; i < B; ++i) {
    sim->flow_base[(size_t)i + 1] = sim->flow_base[(size_t)i] + sim->inst[(size_t)i].n_flows();
    sim->coll_base[(size_t)i + 1] = sim->coll_base[(size_t)i] + (int64_t)sim->inst[(size_t)i].colls.size();
  }
  sim->total_flows = sim->flow_base[(size_t)B];
  sim->total_colls = sim->coll_base[(size_t)B];
  sim->shards.clear();
  sim->shard_first.assign((size_t)n + 1, 0);
  for (int k = 0; k < n; ++k) sim->shard_first[(size_t)k + 1] = sim->shard_first[(size_t)k] + B / n + (k < B % n ? 1 : 0);
  for (int k = 0; k < n; ++k) {
    const int first = sim->shard_first[(size_t)k], cnt = sim->shard_first[(size_t)k + 1] - first;
    std::unique_ptr<phs_sim> c(new phs_sim());
    c->desc = sim->desc;
    c->seed = sim->seed + (uint64_t)first;  // instance i keeps its ECMP seed
    c->batch = cnt;
    c->fab = sim->fab;
    c->inst.assign(sim->inst.begin() + first, sim->inst.begin() + first + cnt);
    c->want_log = sim->want_log;
    c->policy_path = sim->policy_path;
    c->policy_slots = sim->policy_slots;
    c->decompose = sim->decompose;
    c->windows = sim->windows;
    c->hist_cap = sim->hist_cap;
    c->max_snaps = sim->max_snaps;
    c->devices.assign(1, sim->devices[(size_t)k]);
    sim->shards.push_back(std::move(c));
  }
  phs_status st = for_each_shard(sim, [](size_t, phs_sim *c) { return phs_finalize(c, nullptr); });
  if (st != PHS_OK) {
    sim->shards.clear();
    return st;
  }
  sim->h2d_bytes = 0;
  for (const auto &c : sim->shards) sim->h2d_bytes += c->h2d_bytes;
  sim->finalized = true;
  return PHS_OK;
}

}  // namespace

// ================================================================================================ finalize
// Splits the instances into simulation units and builds the device-resident tables.  HBM layout (DESIGN.md "Data
// layout"): one 64-byte FlowRec per flow (path, successors and component inline, unit-local ids), successor lists
// longer than two, predecessor counts (plain and 4-bit packed), the local-flow -> output-position map, per unit
// the capacity row in rate quanta, the link components and the link ids of the topology, the sorted list of
// initial activations, and the dynamic per-flow arrays (pred_cnt, t_done, bneck).
extern "C" phs_status phs_finalize(phs_sim *sim, void *cuda_stream) {
  PHS_API_BEGIN
  if (!sim) return fail(PHS_EINVAL, "null handle");
  if (sim->finalized) return PHS_OK;
  if (sim->devices.size() > 1) return finalize_sharded(sim);
  std::unique_ptr<DeviceGuard> on_device;  // phs_set_devices with one device
  if (sim->devices.size() == 1) on_device.reset(new DeviceGuard(sim->devices[0]));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const bool timing_ = getenv("PHS_TIMING") != nullptr;
  auto tp_ = std::chrono::steady_clock::now();
#define PHS_T(name) if (timing_) { auto n_ = std::chrono::steady_clock::now(); fprintf(stderr, "[phs_finalize] %-22s %8.2f ms\n", name, std::chrono::duration<double, std::milli>(n_ - tp_).count()); tp_ = n_; }
  int dev = 0;
  PHS_CUDA(cudaGetDevice(&dev));
  int sm_count = 0, smem_optin = 0, smem_per_sm = 0;  // three attributes: cudaGetDeviceProperties costs milliseconds
  PHS_CUDA(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev));
  PHS_CUDA(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  PHS_CUDA(cudaDeviceGetAttribute(&smem_per_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev));
  sim->sm_count = sm_count;
  sim->smem_optin = (size_t)smem_optin;
  const int B = sim->batch, L = sim->fab->n_links();

  sim->flow_base.assign(B + 1, 0);
  sim->coll_base.assign(B + 1, 0);
  for (int i = 0; i < B; ++i) {
    sim->flow_base[i + 1] = sim->flow_base[i] + sim->inst[i].n_flows();
    sim->coll_base[i + 1] = sim->coll_base[i] + (int64_t)sim->inst[i].colls.size();
  }
  sim->total_flows = sim->flow_base[B];
  sim->total_colls = sim->coll_base[B];
  const int64_t Ft = sim->total_flows;
  if (Ft >= 0x7fffffffLL) return fail(PHS_ERANGE, "more than 2^31 - 1 flows in one batch");
  const bool split = sim->decompose && !sim->want_log;  // the event log is an instance-wide sequence

  // ---- simulation units (a9).  Flows that share a link, directly or through a chain of flows, and flows joined by
  // a dependency evolve together; such a group shares nothing with the rest of its instance, so (reading R-LZ) it
  // can be simulated on its own with bit-identical results.  Every unit gets dense local flow and link ids.
  // per-instance work is independent: every instance builds its own chunk of the tables on a host thread, the
  // chunks are then laid out back to back
  struct Chunk {
    std::vector<int32_t> succ, lcomp, linkid;
    std::vector<uint8_t> pc8;
    std::vector<int64_t> capq;
    std::vector<double> init_t;
    std::vector<int32_t> init_f;
    std::vector<int32_t> comp_flows, comp_links;  // per component of every unit: flows, links
    std::vector<InstDesc> desc;  // bases relative to the chunk
    std::vector<phs_sim::Unit> units;
    int max_pred = 0;
    phs_status st = PHS_OK;
    const char *err = "";
  };
  std::vector<Chunk> chunks((size_t)B);
  // the per-flow tables (72 of the ~80 bytes per flow) have a known place per instance: the host threads write them
  // straight into the page-locked staging area, unit after unit from flow_base[i] on
  StagingArea &stage = staging_area();
  std::lock_guard<std::mutex> stage_lock(stage.mu);
  const size_t rec_bytes = ((size_t)Ft * sizeof(FlowRec) + 255) / 256 * 256, i32_bytes = ((size_t)Ft * 4 + 255) / 256 * 256;
  unsigned char *stage_p = stage.get(rec_bytes + 2 * i32_bytes);
  if (!stage_p) return fail(PHS_ENOMEM, "out of host memory for the table staging area");
  FlowRec *const rec = (FlowRec *)stage_p;
  int32_t *const pc0 = (int32_t *)(stage_p + rec_bytes);
  uint32_t *const fmap = (uint32_t *)(stage_p + rec_bytes + i32_bytes);
  std::vector<int64_t> coll_first((size_t)sim->total_colls);
  std::vector<int32_t> coll_n((size_t)sim->total_colls);
  auto build_instance = [&](int i) {
    Chunk &c = chunks[(size_t)i];
    expand_pending(*sim->fab, sim->inst[i]);  // a2 + a3 of the collectives submitted since the last expansion
    const Instance &in = sim->inst[i];
    const int64_t F = in.n_flows();
    const int64_t fb = sim->flow_base[i];
    int64_t flow_cursor = 0, log_cursor = 0;
    std::vector<int64_t> capq_inst((size_t)L);
    std::vector<int32_t> parent((size_t)L), uparent((size_t)L), link_loc((size_t)L), link_seen((size_t)L, 0);
    // capacities -> rate quanta (floor); every fair share must stay >= 1 quantum
    for (int l = 0; l < L; ++l) {
      const double cap_l = in.cap.empty() ? sim->fab->default_capacity(l) : in.cap[l];
      const int64_t q = (int64_t)std::floor(cap_l * 1048576.0);
      if (q < F + 1) {
        c.st = PHS_ERANGE;
        c.err = "a link capacity is below (#flows + 1) rate quanta of 2^-20 byte/s";
        return;
      }
      capq_inst[l] = q;
    }
    for (size_t c = 0; c < in.colls.size(); ++c) {
      coll_first[sim->coll_base[i] + c] = sim->flow_base[i] + in.colls[c].first_flow;
      coll_n[sim->coll_base[i] + c] = in.colls[c].n_flows;
    }
    // successor CSR = transpose of the pred lists (counting sort by predecessor)
    std::vector<uint32_t> soff((size_t)F + 1, 0);
    std::vector<int32_t> sdst(in.pred.size());
    for (int32_t p : in.pred) soff[(size_t)p + 1]++;
    for (int64_t f = 0; f < F; ++f) soff[f + 1] += soff[f];
    {
      std::vector<uint32_t> cur(soff.begin(), soff.end() - 1);
      for (int64_t f = 0; f < F; ++f)
        for (uint32_t e = in.pred_off[f]; e < in.pred_off[f + 1]; ++e) sdst[cur[in.pred[e]]++] = (int32_t)f;
    }
    // static link components (union-find over the links, joined by every flow's path; the representative is the
    // smallest link id), and on top of them the units (link components joined by dependencies)
    std::iota(parent.begin(), parent.end(), 0);
    auto find_in = [](std::vector<int32_t> &par, int32_t x) {
      while (par[x] != x) {
        par[x] = par[par[x]];
        x = par[x];
      }
      return x;
    };
    auto unite = [&](std::vector<int32_t> &par, int32_t a, int32_t b) {
      a = find_in(par, a);
      b = find_in(par, b);
      if (a != b) par[std::max(a, b)] = std::min(a, b);
    };
    for (int64_t f = 0; f < F; ++f)
      for (uint32_t e = in.path_off[f] + 1; e < in.path_off[f + 1]; ++e)
        unite(parent, in.path[in.path_off[f]], in.path[e]);
    uparent = parent;
    for (int64_t f = 0; f < F; ++f)
      for (uint32_t e = in.pred_off[f]; e < in.pred_off[f + 1]; ++e)
        unite(uparent, in.path[in.path_off[f]], in.path[in.path_off[in.pred[e]]]);
    // unit of every flow: groups in order of first appearance; groups below 64 flows share bins of up to 256
    std::vector<int32_t> unit_of((size_t)F, 0);
    int32_t n_units = F > 0 ? 1 : 0;
    if (split && F > 0) {
      std::vector<int32_t> group_of_root((size_t)L, -1), gsize;
      for (int64_t f = 0; f < F; ++f) {
        const int32_t r = find_in(uparent, in.path[in.path_off[f]]);
        if (group_of_root[r] < 0) {
          group_of_root[r] = (int32_t)gsize.size();
          gsize.push_back(0);
        }
        unit_of[f] = group_of_root[r];
        gsize[unit_of[f]]++;
      }
      std::vector<int32_t> unit_of_group(gsize.size());
      n_units = 0;
      int32_t bin = -1, bin_flows = 0;
      for (size_t g = 0; g < gsize.size(); ++g) {
        if (gsize[g] >= 64) {
          unit_of_group[g] = n_units++;
        } else {
          if (bin < 0 || bin_flows >= 256) {
            bin = n_units++;
            bin_flows = 0;
          }
          unit_of_group[g] = bin;
          bin_flows += gsize[g];
        }
      }
      for (int64_t f = 0; f < F; ++f) unit_of[f] = unit_of_group[unit_of[f]];
    }
    // flows of every unit in ascending flow id; local flow ids
    std::vector<std::vector<int32_t>> uflows((size_t)n_units);
    std::vector<int32_t> flow_loc((size_t)F);
    for (int64_t f = 0; f < F; ++f) {
      flow_loc[f] = (int32_t)uflows[unit_of[f]].size();
      uflows[unit_of[f]].push_back((int32_t)f);
    }
    // slots a unit can need: raw flows and all-to-alls may be in flight as a whole; a ring collective keeps at most
    // one flow per sender PENDING or ACTIVE, twice the ring size because a slot freed in a phase is reused only in a
    // later one; collectives chained with `after` follow each other per rank, so a chain counts once, with its
    // largest member (a collective and its chain lie in one unit).  The CTA kernel hands a vacated slot straight to
    // the first successor its flow releases, so there a ring of N needs at most N + N/2 slots: N live flows (one
    // per sender) plus one fresh slot per completing flow that releases two successors, and those are at most
    // every second flow of a step (each of the N successors is released once; a flow that releases none queues its
    // slot for the next phase) -- `ubound_cta`.
    std::vector<int64_t> ubound((size_t)n_units, 0), uwhole((size_t)n_units, 0), ubound_cta((size_t)n_units, 0);
    {
      for (int u = 0; u < n_units; ++u) ubound[u] = (int64_t)uflows[u].size();
      for (int u = 0; u < n_units; ++u) uwhole[u] = (int64_t)uflows[u].size();  // minus the ring collectives' flows, below
      for (int u = 0; u < n_units; ++u) ubound_cta[u] = (int64_t)uflows[u].size();
      std::vector<int64_t> chain_max(in.colls.size(), 0), chain_max_cta(in.colls.size(), 0);
      for (size_t c = 0; c < in.colls.size(); ++c) {
        if (in.colls[c].n_flows == 0) continue;
        ubound[unit_of[in.colls[c].first_flow]] -= in.colls[c].n_flows;
        ubound_cta[unit_of[in.colls[c].first_flow]] -= in.colls[c].n_flows;
        const int64_t nr = in.colls[c].n_ranks;
        // chain / tree kinds: one flow per hop (tree edge) and direction is in flight, its successors may be PENDING
        const bool ringk = in.colls[c].kind <= PHS_REDUCESCATTER_RING;
        const int64_t need_cta = in.colls[c].kind == PHS_ALLTOALL
                                     ? in.colls[c].n_flows
                                     : std::min<int64_t>(in.colls[c].n_flows, ringk ? nr + (nr + 1) / 2 : 4 * nr);
        chain_max_cta[in.colls[c].chain] = std::max(chain_max_cta[in.colls[c].chain], need_cta);
        const int64_t need = in.colls[c].kind == PHS_ALLTOALL
                                 ? in.colls[c].n_flows
                                 : std::min<int64_t>(in.colls[c].n_flows, (ringk ? 2 : 4) * (int64_t)in.colls[c].n_ranks);
        chain_max[in.colls[c].chain] = std::max(chain_max[in.colls[c].chain], need);
      }
      for (size_t c = 0; c < in.colls.size(); ++c) {
        if (in.colls[c].n_flows > 0 && in.colls[c].kind != PHS_ALLTOALL)
          uwhole[unit_of[in.colls[c].first_flow]] -= in.colls[c].n_flows;
        if (chain_max[c] > 0) ubound[unit_of[in.colls[c].first_flow]] += chain_max[c];
        if (chain_max_cta[c] > 0) ubound_cta[unit_of[in.colls[c].first_flow]] += chain_max_cta[c];
      }
    }
    // which units hold flows of which collective (ascending per collective), and which flows belong to a collective at
    // all: one pass over the instance, used by the density estimate of every unit below
    std::vector<uint8_t> flow_in_coll((size_t)F, 0);
    std::vector<int32_t> coll_units, coll_units_off(in.colls.size() + 1, 0);
    {
      std::vector<int32_t> seen_by((size_t)std::max(n_units, 1), -1);
      for (size_t ci = 0; ci < in.colls.size(); ++ci) {
        const Collective &co = in.colls[ci];
        for (int32_t f = co.first_flow; f < co.first_flow + co.n_flows; ++f) {
          flow_in_coll[(size_t)f] = 1;
          if (seen_by[(size_t)unit_of[f]] != (int32_t)ci) {
            seen_by[(size_t)unit_of[f]] = (int32_t)ci;
            coll_units.push_back(unit_of[f]);
          }
        }
        std::sort(coll_units.begin() + coll_units_off[ci], coll_units.end());
        coll_units_off[ci + 1] = (int32_t)coll_units.size();
      }
    }
    if (n_units == 0) {  // an instance without flows is one empty unit
      n_units = 1;
      uflows.resize(1);
      ubound.assign(1, 0);
      ubound_cta.assign(1, 0);
      uwhole.assign(1, 0);
    }
    for (int u = 0; u < n_units; ++u) {
      const std::vector<int32_t> &fl = uflows[u];
      // links of the unit, ascending; an undivided instance keeps the whole topology (local id = topology id)
      std::vector<int32_t> links;
      if (n_units == 1) {
        links.resize((size_t)L);
        std::iota(links.begin(), links.end(), 0);
      } else {  // every link once (stamp per link and unit), then ascending: far fewer entries than path hops
        for (int32_t f : fl)
          for (uint32_t e = in.path_off[f]; e < in.path_off[f + 1]; ++e) {
            const int32_t l = in.path[e];
            if (link_seen[(size_t)l] != u + 1) {
              link_seen[(size_t)l] = u + 1;
              links.push_back(l);
            }
          }
        std::sort(links.begin(), links.end());
      }
      for (size_t k = 0; k < links.size(); ++k) link_loc[links[k]] = (int32_t)k;
      InstDesc d;
      d.flow_base = flow_cursor;
      d.link_base = (int64_t)c.capq.size();
      d.succ_base = (int64_t)c.succ.size();
      d.log_base = sim->want_log ? log_cursor : -1;
      d.pc8_base = (int64_t)c.pc8.size();
      d.init_base = (int64_t)c.init_t.size();
      d.n_flows = (int32_t)fl.size();
      d.n_links = (int32_t)links.size();
      // dense component ids, in ascending order of the components' smallest links (links[] is ascending, so a
      // component's representative -- its smallest link -- is met before its other links)
      std::vector<int32_t> comp_id(links.size(), -1);
      int32_t n_comps = 0;
      for (size_t k = 0; k < links.size(); ++k) {
        const int32_t rep = link_loc[find_in(parent, links[k])];
        if (comp_id[rep] < 0) comp_id[rep] = n_comps++;
        comp_id[k] = comp_id[rep];
      }
      d.n_comps = n_comps;
      d.comp_base = (int64_t)c.comp_flows.size();
      c.comp_flows.resize(c.comp_flows.size() + (size_t)n_comps, 0);
      c.comp_links.resize(c.comp_links.size() + (size_t)n_comps, 0);
      int64_t capmax_q = 1;
      for (size_t k = 0; k < links.size(); ++k) {
        c.capq.push_back(capq_inst[links[k]]);
        c.lcomp.push_back(comp_id[k]);
        c.linkid.push_back(links[k]);
        c.comp_links[(size_t)d.comp_base + comp_id[k]]++;
        capmax_q = std::max(capmax_q, capq_inst[links[k]]);
      }
      double lmin = std::numeric_limits<double>::infinity();
      c.pc8.resize(c.pc8.size() + (fl.size() + 7) / 8 * 4, 0);
      for (size_t k = 0; k < fl.size(); ++k) {
        const int32_t f = fl[k];
        FlowRec x;
        x.bytes = in.bytes[f];
        x.start = in.start[f];
        x.lat = in.lat[f];
        const uint32_t p0 = in.path_off[f], p1 = in.path_off[f + 1];
        for (int h = 0; h < kMaxHops; ++h) x.path[h] = p0 + h < p1 ? link_loc[in.path[p0 + h]] : -1;
        x.succ_cnt = (int32_t)(soff[f + 1] - soff[f]);
        if (x.succ_cnt <= 2) {
          x.succ_in[0] = x.succ_cnt > 0 ? flow_loc[sdst[soff[f]]] : -1;
          x.succ_in[1] = x.succ_cnt > 1 ? flow_loc[sdst[soff[f] + 1]] : -1;
        } else {
          x.succ_in[0] = (int32_t)((int64_t)c.succ.size() - d.succ_base);
          x.succ_in[1] = -1;
          for (uint32_t e = soff[f]; e < soff[f + 1]; ++e) c.succ.push_back(flow_loc[sdst[e]]);
        }
        x.comp = p0 < p1 ? comp_id[link_loc[in.path[p0]]] : 0;
        c.comp_flows[(size_t)d.comp_base + x.comp]++;
        rec[(size_t)(fb + flow_cursor) + k] = x;
        fmap[(size_t)(fb + flow_cursor) + k] = (uint32_t)(fb + f);
        const int32_t np = (int32_t)(in.pred_off[f + 1] - in.pred_off[f]);
        if (np > 0) lmin = std::min(lmin, in.lat[f]);
        pc0[(size_t)(fb + flow_cursor) + k] = np;
        c.max_pred = std::max(c.max_pred, np);
        c.pc8[(size_t)d.pc8_base + k / 2] |= (uint8_t)(std::min(np, 15) << ((k & 1) * 4));
      }
      {  // flows without predecessors, by activation time start + Lat (the addition the kernels perform)
        std::vector<std::pair<double, int32_t>> ini;
        for (size_t k = 0; k < fl.size(); ++k)
          if (in.pred_off[fl[k] + 1] == in.pred_off[fl[k]]) ini.emplace_back(in.start[fl[k]] + in.lat[fl[k]], (int32_t)k);
        std::sort(ini.begin(), ini.end());
        d.n_init = (int32_t)ini.size();
        for (const auto &e : ini) {
          c.init_t.push_back(e.first);
          c.init_f.push_back(e.second);
        }
      }
      d.lmin = sim->windows ? lmin : 0.0;
      // Estimated flow events per lookahead window = 2 F lmin / span, with a LOWER bound of the unit's simulated
      // span: every collective takes at least steps x (Lat + chunk / fastest link of the unit), chained collectives
      // follow each other, raw flows at least start + Lat + bytes / fastest link.  Contention only stretches the span,
      // so this over-estimates the density; the window path is worth its per-window overhead only when many events
      // share a window, so a unit goes there when the estimate is well above one (see the scheduler below).
      double density = 0.0;
      if (lmin > 0.0 && !fl.empty()) {
        const double capmax = (double)capmax_q / 1048576.0;
        double span = 0.0;
        std::vector<double> end_of(in.colls.size(), 0.0);
        for (size_t ci = 0; ci < in.colls.size(); ++ci) {
          const Collective &co = in.colls[ci];
          if (co.n_flows == 0) continue;
          // an all-to-all may be split over several units (intra-host / inter-host links)
          const bool here = std::binary_search(coll_units.begin() + coll_units_off[ci],
                                               coll_units.begin() + coll_units_off[ci + 1], (int32_t)u);
          double begin = co.start;
          for (int32_t a : co.after) begin = std::max(begin, end_of[(size_t)a]);
          const double chunk = co.bytes / (double)co.n_ranks;
          end_of[ci] = begin + (double)co.steps * (in.lat[co.first_flow] + chunk / capmax);
          if (here) span = std::max(span, end_of[ci]);
        }
        for (size_t k = 0; k < fl.size(); ++k)
          if (!flow_in_coll[(size_t)fl[k]]) span = std::max(span, in.start[fl[k]] + in.lat[fl[k]] + in.bytes[fl[k]] / capmax);
        density = std::isinf(lmin) ? std::numeric_limits<double>::infinity()
                                   : 2.0 * (double)fl.size() * lmin / std::max(span, 1e-300);
      }
      flow_cursor += (int64_t)fl.size();
      log_cursor += 2 * (int64_t)fl.size() + 2;
      c.desc.push_back(d);
      phs_sim::Unit un;
      un.inst = i;
      un.n_flows = d.n_flows;
      un.n_links = d.n_links;
      un.n_comps = d.n_comps;
      un.bound = ubound[u];
      un.bound_cta = ubound_cta[u];
      un.bound_whole = std::min(ubound[u], uwhole[u]);
      un.comp_base = d.comp_base;
      un.link_base = d.link_base;
      un.density = density;
      un.win_gang = 0;
      c.units.push_back(un);
    }
  };
  PHS_T("setup");
  // The per-flow tables (87 % of the upload) have a known size before anything is built: they get their own device
  // allocation now, and the instances are built in groups so that the finished part of the staging area is already on
  // its way to HBM while the host threads build the next group.
  PHS_CUDA(sim->d_flowtab.alloc(rec_bytes + 2 * i32_bytes));
  sim->d_rec.view((FlowRec *)sim->d_flowtab.p, (size_t)Ft);
  sim->d_pc0.view((int32_t *)(sim->d_flowtab.p + rec_bytes), (size_t)Ft);
  sim->d_fmap.view((uint32_t *)(sim->d_flowtab.p + rec_bytes + i32_bytes), (size_t)Ft);
  {
    const int n_groups = std::max(1, std::min(8, B / 64));
    for (int g = 0; g < n_groups; ++g) {
      const int i0 = (int)((int64_t)B * g / n_groups), i1 = (int)((int64_t)B * (g + 1) / n_groups);
      parallel_for(i1 - i0, [&](int k) { build_instance(i0 + k); });
      const size_t f0 = (size_t)sim->flow_base[i0], nf = (size_t)(sim->flow_base[i1] - sim->flow_base[i0]);
      if (nf == 0) continue;
      PHS_CUDA(cudaMemcpyAsync(sim->d_rec.p + f0, rec + f0, nf * sizeof(FlowRec), cudaMemcpyHostToDevice, st));
      PHS_CUDA(cudaMemcpyAsync(sim->d_pc0.p + f0, pc0 + f0, nf * sizeof(int32_t), cudaMemcpyHostToDevice, st));
      PHS_CUDA(cudaMemcpyAsync(sim->d_fmap.p + f0, fmap + f0, nf * sizeof(uint32_t), cudaMemcpyHostToDevice, st));
    }
  }
  PHS_T("build_instances");
  for (int i = 0; i < B; ++i)
    if (chunks[i].st != PHS_OK) return fail(chunks[i].st, chunks[i].err);
  // lay the chunks out back to back
  std::vector<int64_t> b_flow(B + 1, 0), b_link(B + 1, 0), b_succ(B + 1, 0), b_pc8(B + 1, 0), b_log(B + 1, 0),
      b_init(B + 1, 0), b_comp(B + 1, 0);
  sim->units.clear();
  sim->unit_first.assign(B + 1, 0);
  int max_pred = 0;
  for (int i = 0; i < B; ++i) {
    const Chunk &c = chunks[i];
    b_flow[i + 1] = sim->flow_base[i + 1];
    b_link[i + 1] = b_link[i] + (int64_t)c.capq.size();
    b_succ[i + 1] = b_succ[i] + (int64_t)c.succ.size();
    b_pc8[i + 1] = b_pc8[i] + (int64_t)c.pc8.size();
    b_init[i + 1] = b_init[i] + (int64_t)c.init_t.size();
    b_comp[i + 1] = b_comp[i] + (int64_t)c.comp_flows.size();
    b_log[i + 1] = b_log[i] + 2 * (sim->flow_base[i + 1] - sim->flow_base[i]) + 2 * (int64_t)c.units.size();
    sim->unit_first[i] = (int32_t)sim->units.size();
    sim->units.insert(sim->units.end(), c.units.begin(), c.units.end());
    for (size_t k = sim->units.size() - c.units.size(); k < sim->units.size(); ++k) {
      sim->units[k].comp_base += b_comp[i];
      sim->units[k].link_base += b_link[i];
    }
    max_pred = std::max(max_pred, c.max_pred);
  }
  const int64_t log_cursor = b_log[B];
  std::vector<int32_t> succ((size_t)b_succ[B]), lcomp((size_t)b_link[B]), linkid((size_t)b_link[B]);
  std::vector<uint8_t> pc8((size_t)b_pc8[B]);
  std::vector<int64_t> capq((size_t)b_link[B]);
  std::vector<double> init_t((size_t)b_init[B]);
  std::vector<int32_t> init_f((size_t)b_init[B]);
  sim->h_desc.assign(sim->units.size(), InstDesc{});
  sim->comp_flows.assign((size_t)b_comp[B], 0);
  sim->comp_links.assign((size_t)b_comp[B], 0);
  parallel_for(B, [&](int i) {
    Chunk &c = chunks[i];
    std::copy(c.comp_flows.begin(), c.comp_flows.end(), sim->comp_flows.begin() + b_comp[i]);
    std::copy(c.comp_links.begin(), c.comp_links.end(), sim->comp_links.begin() + b_comp[i]);
    std::copy(c.succ.begin(), c.succ.end(), succ.begin() + b_succ[i]);
    std::copy(c.pc8.begin(), c.pc8.end(), pc8.begin() + b_pc8[i]);
    std::copy(c.capq.begin(), c.capq.end(), capq.begin() + b_link[i]);
    std::copy(c.lcomp.begin(), c.lcomp.end(), lcomp.begin() + b_link[i]);
    std::copy(c.linkid.begin(), c.linkid.end(), linkid.begin() + b_link[i]);
    std::copy(c.init_t.begin(), c.init_t.end(), init_t.begin() + b_init[i]);
    std::copy(c.init_f.begin(), c.init_f.end(), init_f.begin() + b_init[i]);
    for (size_t k = 0; k < c.desc.size(); ++k) {
      InstDesc d = c.desc[k];
      d.flow_base += b_flow[i];
      d.link_base += b_link[i];
      d.succ_base += b_succ[i];
      d.pc8_base += b_pc8[i];
      d.init_base += b_init[i];
      d.comp_base += b_comp[i];
      if (d.log_base >= 0) d.log_base += b_log[i];
      sim->h_desc[(size_t)sim->unit_first[i] + k] = d;
    }
  });
  PHS_T("concat");
  sim->unit_first[B] = (int32_t)sim->units.size();
  const int U = (int)sim->units.size();
  // window path (a9): which units run the lookahead-window schedule, and the ownership tables of their gangs
  sim->h_lcomp = lcomp;
  sim->h_lloc.assign(lcomp.size(), 0);
  sim->h_cown.assign((size_t)b_comp[B], 0);
  sim->win_list.clear();
  for (int u = 0; u < U; ++u)
    if (plan_window_unit(sim, u, (size_t)smem_optin, sim->win_scale)) sim->win_list.push_back(u);
  PHS_T("window plan");
  const bool pc8_ok = max_pred <= 15;  // the packed counters hold 4 bits per flow

  // one device allocation for all other tables and the result arrays (a cudaMalloc costs about 0.1 ms, and there are
  // 16 of them): first pass sizes, second pass places the views and issues the copies
  {
    unsigned char *base = nullptr;
    size_t cursor = 0;
    cudaError_t err = cudaSuccess;
    auto put = [&](auto &buf, const auto *h, size_t count) {
      using T = typename std::remove_pointer<decltype(buf.p)>::type;
      if (base) {
        buf.view((T *)(base + cursor), count);
        if (h && count && err == cudaSuccess)
          err = cudaMemcpyAsync(buf.p, h, count * sizeof(T), cudaMemcpyHostToDevice, st);
      }
      cursor += (std::max<size_t>(count, 1) * sizeof(T) + 255) / 256 * 256;
    };
    auto put_all = [&] {
      cursor = 0;
      put(sim->d_desc, sim->h_desc.data(), sim->h_desc.size());
      if (pc8_ok) put(sim->d_pc8, pc8.data(), pc8.size());
      put(sim->d_succ, succ.data(), succ.size());
      put(sim->d_init_t, init_t.data(), init_t.size());
      put(sim->d_init_f, init_f.data(), init_f.size());
      put(sim->d_capq, capq.data(), capq.size());
      put(sim->d_lcomp, lcomp.data(), lcomp.size());
      put(sim->d_linkid, linkid.data(), linkid.size());
      put(sim->d_coll_first, coll_first.data(), coll_first.size());
      put(sim->d_coll_n, coll_n.data(), coll_n.size());
      put(sim->d_pred_cnt, (const int32_t *)nullptr, (size_t)Ft);
      put(sim->d_tdone, (const double *)nullptr, (size_t)Ft);
      put(sim->d_bneck, (const int32_t *)nullptr, (size_t)Ft);
      put(sim->d_coll_t, (const double *)nullptr, (size_t)sim->total_colls);
      put(sim->d_res, (const InstResult *)nullptr, (size_t)U);
      put(sim->d_ticket, (const int *)nullptr, 1);
    };
    put_all();
    PHS_CUDA(sim->d_arena.alloc(cursor));
    base = sim->d_arena.p;
    put_all();
    PHS_CUDA(err);
  }
  PHS_CUDA(sim->d_lloc.upload(sim->h_lloc, st));
  PHS_CUDA(sim->d_cown.upload(sim->h_cown, st));
  if (sim->want_log) PHS_CUDA(sim->d_log.alloc((size_t)log_cursor));
  if (sim->hist_cap > 0) {
    PHS_CUDA(sim->d_hist.alloc((size_t)sim->hist_cap));
    PHS_CUDA(sim->d_hist_n.alloc(1));
  }
  sim->h_res.assign(U, InstResult{});
  PHS_T("upload+alloc issued");

  // ---- a9: batch scheduler, static part.  A unit whose state fits the shared memory of one SM goes to the CTA
  // path (one launch configuration, sized for the largest such unit, with as many CTAs resident per SM as fit);
  // the others go to the cluster path.  Units that overflow their slots at run time move to the cluster path.
  const size_t smem_max = (size_t)smem_optin;
  const size_t per_sm = (size_t)smem_per_sm;
  const bool log = sim->want_log;
  sim->order.clear();
  sim->cluster_list.clear();
  sim->grid_list.clear();
  sim->cta = CtaLaunch{};
  auto need_of = [&](const phs_sim::Unit &u) {
    return (int)std::min<int64_t>(std::min<int64_t>(std::max<int64_t>(u.n_flows, 1), std::max<int64_t>(u.bound_cta, 32)), 1 << 16);
  };
  std::vector<int32_t> cand;
  for (int u = 0; u < U; ++u) {
    const phs_sim::Unit &un = sim->units[u];
    if (un.n_flows == 0) continue;  // nothing to simulate; its result block stays zero (status OK)
    if (un.win_gang > 0) continue;  // runs on the window path
    if (sim->policy_path == 4 && !log) {  // phs_set_scheduler: the whole grid for every unit
      sim->grid_list.push_back(u);
      continue;
    }
    if (sim->policy_path == 2 || un.n_links >= 65535 ||
        cta_smem_bytes(un.n_links, (need_of(un) + 31) / 32 * 32, 0, log) > smem_max)
      sim->cluster_list.push_back(u);
    else
      cand.push_back(u);
  }
  while (!cand.empty()) {
    int Lm = 1, NCm = 1, need = 32;
    int64_t maxF = 1;
    for (int u : cand) {
      Lm = std::max(Lm, sim->units[u].n_links);
      NCm = std::max(NCm, sim->units[u].n_comps);
      need = std::max(need, need_of(sim->units[u]));
      maxF = std::max<int64_t>(maxF, sim->units[u].n_flows);
    }
    // about one slot per thread: measured on B200, 128 threads for cfg3-sized units, 256 for cfg1-sized ones
    // about one slot per thread makes one unit's event shortest (cfg1, bound by its 64 longest units: 256 threads
    // 10.8 ms, 128 threads 12.5 ms, 64 threads 15.9 ms).  With many times more units than can be resident the SMs'
    // issue slots are the limit, not the length of one event, and half as many threads waste fewer of them (cfg3,
    // 36,864 units: 128 threads 57 ms, 64 threads 47 ms, 32 threads 58 ms).  Measured on B200.
    int threads = (need <= 128 && Lm <= 320) ? 128 : 256;
    if ((int64_t)cand.size() >= 64LL * sim->sm_count) threads /= 2;
    if (const char *ev = getenv("PHS_CTA_THREADS")) {  // tuning experiments; anything but a supported size is ignored
      const int v = atoi(ev);
      if (v == 32 || v == 64 || v == 128 || v == 256 || v == 512) threads = v;
    }
    const int want = std::max(1, std::min(2048 / threads / 2, ((int)cand.size() + sim->sm_count - 1) / sim->sm_count));
    // largest number of resident CTAs per SM (<= want) whose shared memory holds `need` slots, with or without the
    // predecessor counters on chip; returns 0 if not even one fits
    auto fit = [&](bool pcs, int lean, int *slots_out) {
      const int pcf = pcs ? (int)maxF : 0;
      for (int w = want; w >= 1; --w) {
        const size_t budget = std::min(smem_max, per_sm / w - 1024);
        if (cta_smem_bytes(Lm, 32, pcf, log, lean) > budget) continue;
        int lo = 32, hi = (int)std::min<int64_t>(std::max<int64_t>(maxF, 32), 1 << 16);
        if (sim->policy_slots > 0 && sim->policy_path != 3) hi = std::max(32, std::min(hi, (int)sim->policy_slots));
        hi = (hi + 31) / 32 * 32;
        while (lo < hi) {  // largest multiple of 32 that fits the budget
          const int mid = ((lo + hi + 32) / 64) * 32;
          if (cta_smem_bytes(Lm, mid, pcf, log, lean) <= budget)
            lo = mid;
          else
            hi = mid - 32;
        }
        const bool capped = sim->policy_slots > 0 && sim->policy_path != 3;
        if (lo >= need || (w == 1 && sim->policy_path == 1) || capped) {
          if (!capped) lo = std::min(lo, (need + 31) / 32 * 32);  // no more than can be used
          *slots_out = lo;
          return w;
        }
      }
      return 0;
    };
    // Lean layout (CtaLaunch::lean): in the throughput regime (the same test as for the thread count) every further
    // resident CTA hides latency, so the per-link arrays that only multi-round solves touch -- and, if that buys
    // another CTA, the capacities -- leave shared memory.  Latency-bound batches keep everything on chip.
    int lean = 0;
    if ((int64_t)cand.size() >= 64LL * sim->sm_count && !log) {
      int best_w = 0;
      for (int cand_lean : {0, 1, 3}) {
        int sl = 0;
        const int w = std::max(pc8_ok ? fit(true, cand_lean, &sl) : 0, fit(false, cand_lean, &sl));
        if (w > best_w) {
          best_w = w;
          lean = cand_lean;
        }
      }
    }
    if (const char *ev = getenv("PHS_CTA_LEAN")) {  // tuning experiments
      const int v = atoi(ev);
      if (v == 0 || v == 1 || v == 3) lean = log ? 0 : v;
    }
    // Incremental re-solve (bit 2 of `lean`): where most of the launch's flows are all-to-all or raw
    // flow sets -- solves of several filling rounds -- and nothing else claims the working arrays (no lean layout, no
    // event log, no history).  Ring traffic solves in one round and is better off without it.
    {
      int64_t whole = 0, all = 0;
      for (int u : cand) {
        whole += std::min<int64_t>(sim->units[u].bound_whole, sim->units[u].n_flows);
        all += sim->units[u].n_flows;
      }
      bool inc = lean == 0 && !log && sim->hist_cap == 0 && 2 * whole >= all;
      if (const char *ev = getenv("PHS_CTA_INC")) inc = atoi(ev) != 0 && lean == 0 && !log && sim->hist_cap == 0;
      if (inc) lean = 4;
    }
    int slots_p = 0, slots_n = 0;
    const int w_p = pc8_ok ? fit(true, lean, &slots_p) : 0, w_n = fit(false, lean, &slots_n);
    if (w_p == 0 && w_n == 0) {
      // the largest links x slots combination does not fit one SM: the unit with the most flows goes to a cluster
      auto big = std::max_element(cand.begin(), cand.end(), [&](int a, int b) {
        return sim->units[a].n_flows < sim->units[b].n_flows;
      });
      sim->cluster_list.push_back(*big);
      cand.erase(big);
      continue;
    }
    // counters on chip save an L2 round trip per release: worth one resident CTA less
    const bool pcs = w_p > 0 && slots_p >= std::min(need, slots_n) && w_p >= w_n - 1;
    sim->cta.threads = threads;
    sim->cta.slots = pcs ? slots_p : slots_n;
    sim->cta.pc_flows = pcs ? (int)maxF : 0;
    sim->cta.smem = cta_smem_bytes(Lm, sim->cta.slots, sim->cta.pc_flows, log, lean);
    sim->cta.lean = lean;
    sim->cta.lean_scratch = nullptr;  // allocated below, once the grid is known
    sim->cta.log = log;
    sim->cta.n_links = Lm;
    sim->order = cand;
    std::stable_sort(sim->order.begin(), sim->order.end(),
                     [&](int a, int b) { return sim->units[a].n_flows > sim->units[b].n_flows; });
    const int per = std::max(1, std::min<int>((int)(per_sm / (sim->cta.smem + 1024)), 2048 / threads));
    sim->cta.grid = std::min((int)cand.size(), per * sim->sm_count);
    PHS_CUDA(sim->d_order.upload(sim->order, st));
    if (lean & 1) {
      PHS_CUDA(sim->d_lean.alloc(cta_lean_scratch_bytes(Lm) * (size_t)sim->cta.grid));
      sim->cta.lean_scratch = sim->d_lean.p;
    }
    if (timing_)
      fprintf(stderr, "[phs_finalize] cta path: %d units, threads %d, need %d, links %d, slots %d, smem %zu, lean %d, grid %d (%d per SM)\n",
              (int)cand.size(), threads, need, Lm, sim->cta.slots, sim->cta.smem, lean, sim->cta.grid, per);
    break;
  }
  std::sort(sim->cluster_list.begin(), sim->cluster_list.end());
  PHS_T("scheduler");
  PHS_CUDA(cudaStreamSynchronize(st));  // the staging vectors die here
  PHS_T("sync");
  sim->h2d_bytes = (int64_t)(sim->h_desc.size() * sizeof(InstDesc) + (size_t)Ft * sizeof(FlowRec) +
                             (succ.size() + (size_t)Ft + coll_n.size() + sim->order.size() + lcomp.size() + linkid.size() +
                              (size_t)Ft + init_f.size()) * 4 + init_t.size() * 8 + (pc8_ok ? pc8.size() : 0) +
                             (capq.size() + coll_first.size()) * 8);
  PHS_CUDA(cudaEventCreate(&sim->ev0));
  PHS_CUDA(cudaEventCreate(&sim->ev1));
  sim->finalized = true;
  return PHS_OK;
  PHS_API_END
}

// ================================================================================================ run
namespace {

DevTables tables_of(phs_sim *sim, int n_links) {
  DevTables t;
  t.lloc = sim->d_lloc.p;
  t.cown = sim->d_cown.p;
  t.t_rel = sim->d_trel.p;
  t.fcw = sim->d_fcw.p;
  t.inst = sim->d_desc.p;
  t.rec = sim->d_rec.p;
  t.succ = sim->d_succ.p;
  t.pred_cnt0 = sim->d_pc0.p;
  t.pred_cnt0_u8 = sim->d_pc8.p;
  t.fmap = sim->d_fmap.p;
  t.init_t = sim->d_init_t.p;
  t.init_f = sim->d_init_f.p;
  t.capq = sim->d_capq.p;
  t.lcomp = sim->d_lcomp.p;
  t.linkid = sim->d_linkid.p;
  t.pred_cnt = sim->d_pred_cnt.p;
  t.t_done = sim->d_tdone.p;
  t.bneck = sim->d_bneck.p;
  t.res = sim->d_res.p;
  t.log = sim->want_log ? sim->d_log.p : nullptr;
  t.hist = sim->hist_cap > 0 ? sim->d_hist.p : nullptr;
  t.hist_n = sim->d_hist_n.p;
  t.hist_cap = sim->hist_cap;
  t.t_stop = sim->t_stop;
  t.park = nullptr;  // set by phs_run_until for the CTA path
  t.park_stride = 0;
  t.resume = 0;
  t.n_links = n_links;
  return t;
}

// Cluster path (a9): every instance in `list` is simulated by one thread-block cluster with all dynamic state in
// the shared memory of its CTAs; clusters pull instances from the list until it is empty.  `slot_scale` scales the
// guess of how many flows are PENDING or ACTIVE at once (doubled after an overflow).
phs_status run_cluster_path(phs_sim *sim, std::vector<int32_t> list, int64_t slot_scale, bool park, bool resume,
                            cudaStream_t st, std::vector<int32_t> *too_big) {
retry:
  if (list.empty()) return PHS_OK;
  // The launch configuration is sized for ALL units of the cluster path, not only the ones of this call (a resume
  // runs the unfinished ones): parked states and snapshots stay valid from call to call.
  std::vector<int32_t> basis(sim->cluster_list);
  for (int u : list)
    if (std::find(basis.begin(), basis.end(), u) == basis.end()) basis.push_back(u);
  for (int u : *too_big) basis.erase(std::remove(basis.begin(), basis.end(), u), basis.end());
  int L = 1;  // the shared-memory layout is sized for the unit with the most links
  for (int u : basis) L = std::max(L, sim->units[u].n_links);
  if (L >= 65535) return fail(PHS_ERANGE, "cluster path: units with 65535 or more links are not supported");
  // slots needed per instance: every flow without predecessors is PENDING from t = 0; later, a ring collective
  // has at most one step in flight per rank plus the successors waiting out their latency, while an all-to-all
  // or a raw flow set can be in flight as a whole.  Start from a quarter of that bound; overflow doubles it.
  int64_t target = 64;
  for (int u : basis) {
    const phs_sim::Unit &un = sim->units[u];
    const int64_t ring = un.bound - un.bound_whole;  // rarely all in flight at once: start from a quarter
    target = std::max(target, un.bound_whole + std::min(ring, ring * slot_scale / 4));
    if (slot_scale > 4) target = std::max(target, std::min<int64_t>(un.n_flows, un.bound * slot_scale / 4));
  }
  const size_t smem_max = sim->smem_optin - 4096;  // minus the kernel's static shared memory
  const bool log = sim->want_log;
  int cs = 0, max_clusters = 0;
  int64_t Sc = 0;
  bool agg = false, cold = false, repl = false;
  // replicated link shares pay when many flows share a link (every flow reads its links' shares every round)
  const bool want_repl = target >= 8 * (int64_t)L;
  for (int c = 1; c <= 16 && !cs; c *= 2) {
    if ((int64_t)c * kClusterThreads * 4 < target && c < 16) continue;  // at most ~4 slots per thread
    const int64_t sc = std::min<int64_t>(65535, (target + c - 1) / c + 16);
    const bool opts[4][2] = {{true, true}, {false, true}, {true, false}, {false, false}};  // {agg, cold in smem}
    for (int k = 0; k < 8 && !cs; ++k) {
      const bool o_agg = opts[k & 3][0], o_cold = opts[k & 3][1], o_repl = k < 4;
      if (o_repl && !want_repl) continue;
      if (c < 16 && !o_cold) continue;  // spill cold fields to global only at the largest cluster size
      const size_t smem = cluster_smem_bytes(L, c, sc, o_agg, o_cold, log, o_repl);
      if (smem > smem_max) continue;
      int n = 0;
      PHS_CUDA(cluster_max_clusters(c, smem, &n));
      if (n < 1) continue;
      cs = c;
      Sc = sc;
      agg = o_agg;
      cold = o_cold;
      repl = o_repl;
      max_clusters = n;
    }
  }
  if (!cs) {
    // the unit with the most concurrent flows fits no cluster: the whole grid simulates it, with its state in global
    // memory (grid path); the event log is not written there
    if (log)
      return fail(PHS_ERANGE, "a unit's pending + active flows do not fit the shared memory of a cluster, and the grid "
                              "path does not write the event log");
    auto big = std::max_element(basis.begin(), basis.end(), [&](int a, int b) {
      const phs_sim::Unit &x = sim->units[(size_t)a], &y = sim->units[(size_t)b];
      return x.bound_whole + (x.bound - x.bound_whole) / 4 < y.bound_whole + (y.bound - y.bound_whole) / 4;
    });
    too_big->push_back(*big);
    list.erase(std::remove(list.begin(), list.end(), *big), list.end());
    goto retry;
  }
  const int n_clusters = std::max(1, std::min<int>((int)list.size(), max_clusters));
  const size_t region = cold ? 0 : cluster_region_bytes(Sc, cs);
  if (region * n_clusters > sim->g_scratch.n) PHS_CUDA(sim->g_scratch.alloc(region * n_clusters));
  if (!sim->d_cticket.p) PHS_CUDA(sim->d_cticket.alloc(1));
  sim->scratch_Sc = Sc;
  sim->scratch_cs = cs;
  sim->clusters_resident = max_clusters;
  std::vector<int32_t> sorted(list);
  std::stable_sort(sorted.begin(), sorted.end(),
                   [&](int a, int b) { return sim->units[a].n_flows > sim->units[b].n_flows; });
  PHS_CUDA(sim->d_clist.upload(sorted, st));
  PHS_CUDA(cudaMemsetAsync(sim->d_cticket.p, 0, sizeof(int), st));
  ClusterScratch sc;
  sc.base = sim->g_scratch.p;
  sc.region_bytes = region;
  sc.Sc = Sc;
  sc.aggregate = agg ? 1 : 0;
  sc.cold_smem = cold ? 1 : 0;
  sc.replicate = repl ? 1 : 0;
  sc.incremental = (repl && agg && !log) ? 1 : 0;
  if (const char *ev = getenv("PHS_CLUSTER_INC")) sc.incremental = (atoi(ev) != 0 && repl && agg && !log) ? 1 : 0;  // tuning
  // phs_run_until: parking areas, one per cluster-path unit, valid for one launch configuration
  sc.park = nullptr;
  sc.park_unit_stride = sc.park_cta_stride = 0;
  sc.park_index = nullptr;
  sc.resume = 0;
  if (park || resume) {
    const size_t cta_bytes = cluster_park_cta_bytes(L, cs, Sc, agg, cold, log, repl);
    const size_t unit_bytes = kClusterParkHeader + (size_t)cs * cta_bytes;
    const bool same = sim->cpark_unit_bytes == unit_bytes && sim->cpark_cs == cs && sim->cpark_Sc == Sc &&
                      sim->cpark_L == L && sim->d_cpark.p;
    if (!same) {  // (re)build: every unit of the cluster list gets an area; what was parked before is void
      std::vector<int32_t> index(sim->units.size(), -1);
      int32_t n = 0;
      for (int u : sim->cluster_list) index[u] = n++;
      for (int u : list)
        if (index[u] < 0) index[u] = n++;
      PHS_CUDA(sim->d_cpark.alloc(unit_bytes * (size_t)std::max(n, 1)));
      PHS_CUDA(cudaMemsetAsync(sim->d_cpark.p, 0, unit_bytes * (size_t)std::max(n, 1), st));
      PHS_CUDA(sim->d_cpark_index.upload(index, st));
      PHS_CUDA(cudaStreamSynchronize(st));
      sim->cpark_index = index;
      sim->cpark_unit_bytes = unit_bytes;
      sim->cpark_cs = cs;
      sim->cpark_Sc = Sc;
      sim->cpark_L = L;
    }
    bool all_indexed = true;
    for (int u : list) all_indexed = all_indexed && sim->cpark_index[u] >= 0;
    if (all_indexed) {  // units that joined the cluster path later (slot overflow) simply start from t = 0
      sc.park = sim->d_cpark.p;
      sc.park_unit_stride = unit_bytes;
      sc.park_cta_stride = cta_bytes;
      sc.park_index = sim->d_cpark_index.p;
      sc.resume = resume && same ? 1 : 0;
    }
  }
  PHS_CUDA(launch_cluster_path(tables_of(sim, L), sim->d_clist.p, (int)sorted.size(), sim->d_cticket.p, sc, cs,
                               n_clusters, log, st));
  PHS_CUDA(cudaStreamSynchronize(st));  // `sorted` is pageable host memory read by the async copy
  return PHS_OK;
}


// Grid path (a9): the whole grid (cooperative launch) simulates the units of `list` one after the other.
phs_status run_grid_path(phs_sim *sim, const std::vector<int32_t> &list, cudaStream_t st) {
  if (list.empty()) return PHS_OK;
  int64_t Fm = 1;
  int Lm = 1;
  for (int u : list) {
    Fm = std::max<int64_t>(Fm, sim->units[(size_t)u].n_flows);
    Lm = std::max(Lm, sim->units[(size_t)u].n_links);
  }
  const size_t bytes = grid_scratch_bytes(Fm, Lm);
  PHS_DBG("grid path: %d units, Fm %lld Lm %d scratch %zu", (int)list.size(), (long long)Fm, Lm, bytes);
  if (bytes > sim->d_gscratch.n) PHS_CUDA(sim->d_gscratch.alloc(bytes));
  int n_ctas = 0;
  PHS_CUDA(grid_max_ctas(&n_ctas));
  PHS_DBG("grid path: max ctas %d", n_ctas);
  if (n_ctas < 1) return fail(PHS_ECUDA, "grid path: the kernel cannot be resident");
  // no more CTAs than the largest unit can use (one flow per thread)
  n_ctas = (int)std::max<int64_t>(1, std::min<int64_t>(n_ctas, (Fm + kGridThreads - 1) / kGridThreads));
  if (const char *ev = getenv("PHS_GRID_CTAS")) {  // tuning experiments: fewer CTAs than the default
    const int v = atoi(ev);
    if (v >= 1 && v < n_ctas) n_ctas = v;
  }
  PHS_CUDA(sim->d_glist.upload(list, st));
  PHS_CUDA(launch_grid_path(tables_of(sim, Lm), sim->d_glist.p, (int)list.size(), sim->d_gscratch.p, Fm, Lm, n_ctas, st));
  PHS_DBG("grid path: launched");
  PHS_CUDA(cudaStreamSynchronize(st));  // `list` may be pageable host memory read by the async copy
  PHS_DBG("grid path: done");
  sim->grid_ctas = n_ctas;
  sim->n_launches++;
  return PHS_OK;
}

// Window path (a9): the units of `todo` run the lookahead-window schedule, one gang of CTAs each; gangs of one size
// share a launch.  Units that run out of slots are planned again with a larger estimate (possibly a larger gang);
// the ones that do not fit any more are returned in `fallback` (they go to the cluster path).
phs_status run_window_path(phs_sim *sim, std::vector<int32_t> todo, std::vector<int32_t> *fallback, cudaStream_t st) {
  if (!sim->d_wticket.p) PHS_CUDA(sim->d_wticket.alloc(1));
  if (!sim->d_trel.p) {  // per-flow scratch of the window path (initialised by the kernel, unit by unit)
    PHS_CUDA(sim->d_trel.alloc((size_t)sim->total_flows));
    PHS_CUDA(sim->d_fcw.alloc((size_t)sim->total_flows));
  }
  int64_t scale = sim->win_scale;
  while (!todo.empty()) {
    for (int K = 1; K <= 16; K *= 2) {
      std::vector<int32_t> group;
      for (int u : todo)
        if (sim->units[(size_t)u].win_gang == K) group.push_back(u);
      // one launch per set of units whose combined layout (largest links, components, slots per CTA) fits
      std::stable_sort(group.begin(), group.end(),
                       [&](int a, int b) { return sim->units[(size_t)a].n_flows > sim->units[(size_t)b].n_flows; });
      size_t pos = 0;
      while (pos < group.size()) {
        WindowLaunch w{};
        w.gang = K;
        size_t end = pos;
        for (; end < group.size(); ++end) {
          const phs_sim::Unit &un = sim->units[(size_t)group[end]];
          const int L2 = std::max(w.n_links, un.win_links), C2 = std::max(w.n_comps, un.win_comps),
                    S2 = std::max(w.slots, un.win_slots);
          if (end > pos && window_smem_bytes(L2, C2, S2) + 512 > sim->smem_optin) break;
          w.n_links = L2;
          w.n_comps = C2;
          w.slots = S2;
        }
        w.smem = window_smem_bytes(w.n_links, w.n_comps, w.slots);
        std::vector<int32_t> part(group.begin() + (long)pos, group.begin() + (long)end);
        int max_clusters = 0;
        PHS_CUDA(window_max_clusters(K, w.smem, &max_clusters));
        if (max_clusters < 1) return fail(PHS_ECUDA, "window path: a gang of " + std::to_string(K) + " CTAs cannot be resident");
        const int n_clusters = std::min<int>((int)part.size(), max_clusters);
        PHS_CUDA(sim->d_wlist.upload(part, st));
        PHS_CUDA(cudaMemsetAsync(sim->d_wticket.p, 0, sizeof(int), st));
        int Lmax = 1;
        for (int u : part) Lmax = std::max(Lmax, sim->units[(size_t)u].n_links);
        if (getenv("PHS_TIMING"))
          fprintf(stderr, "[phs_run] window path: %d units, gang %d, per CTA: links %d, comps %d, slots %d, smem %zu; %d gangs resident\n",
                  (int)part.size(), K, w.n_links, w.n_comps, w.slots, w.smem, n_clusters);
        PHS_CUDA(launch_window_path(tables_of(sim, Lmax), sim->d_wlist.p, (int)part.size(), sim->d_wticket.p, w,
                                    n_clusters, st));
        PHS_CUDA(cudaStreamSynchronize(st));  // `part` is pageable host memory read by the async copy
        sim->n_launches++;
        sim->win_gang_used = std::max(sim->win_gang_used, K);
        pos = end;
      }
    }
    const int U = (int)sim->units.size();
    PHS_CUDA(cudaMemcpyAsync(sim->h_res.data(), sim->d_res.p, sizeof(InstResult) * U, cudaMemcpyDeviceToHost, st));
    PHS_CUDA(cudaStreamSynchronize(st));
    std::vector<int32_t> again;
    for (int u : todo)
      if (sim->h_res[(size_t)u].status == kOverflow) again.push_back(u);
    if (again.empty()) break;
    scale *= 2;  // more slots, possibly a larger gang; what does not fit any more leaves the window path for good
    sim->win_scale = scale;
    todo.clear();
    for (int u : again) {
      if (scale <= 64 && plan_window_unit(sim, u, sim->smem_optin, scale)) {
        todo.push_back(u);
      } else {
        sim->units[(size_t)u].win_gang = 0;
        sim->win_list.erase(std::find(sim->win_list.begin(), sim->win_list.end(), u));
        fallback->push_back(u);
      }
    }
    PHS_CUDA(sim->d_lloc.upload(sim->h_lloc, st));
    PHS_CUDA(sim->d_cown.upload(sim->h_cown, st));
    PHS_CUDA(cudaStreamSynchronize(st));
  }
  return PHS_OK;
}

}  // namespace


// ================================================================================================ NEXT-1: rollback
void phs_unfinalize(phs_sim *sim) {
  sim->finalized = sim->ran = sim->have_park = false;
  sim->snaps.clear();
  sim->dirty_from = std::numeric_limits<double>::infinity();
  sim->h_pos.clear();
  sim->park_stride = 0;
  sim->cpark_unit_bytes = 0;
  sim->cpark_cs = sim->cpark_L = 0;
  sim->cpark_Sc = 0;
  sim->d_park.release();
  sim->d_cpark.release();
  sim->d_cpark_index.release();
  sim->d_trel.release();
  sim->d_fcw.release();
  sim->d_hist.release();
  sim->d_hist_n.release();
  sim->d_log.release();
  sim->d_arena.release();  // the table buffers are views into it
  sim->d_flowtab.release();  // ... and the per-flow tables into this one
  if (sim->ev0) cudaEventDestroy(sim->ev0);
  if (sim->ev1) cudaEventDestroy(sim->ev1);
  sim->ev0 = sim->ev1 = nullptr;
}

namespace {

// keeps the parked state of the run that just stopped at sim->parked_until (newest last, at most max_snaps)
phs_status take_snapshot(phs_sim *sim, cudaStream_t st) {
  if (sim->max_snaps <= 0 || !sim->have_park) return PHS_OK;
  if (!sim->snaps.empty() && sim->snaps.back()->t == sim->parked_until) return PHS_OK;
  std::unique_ptr<phs_sim::Snapshot> sn(new phs_sim::Snapshot());
  sn->t = sim->parked_until;
  if (sim->d_park.p && sim->park_stride) {
    const size_t n = sim->park_stride * sim->units.size();
    PHS_CUDA(sn->park.alloc(n));
    PHS_CUDA(cudaMemcpyAsync(sn->park.p, sim->d_park.p, n, cudaMemcpyDeviceToDevice, st));
  }
  if (sim->d_cpark.p && sim->d_cpark.n) {
    PHS_CUDA(sn->cpark.alloc(sim->d_cpark.n));
    PHS_CUDA(cudaMemcpyAsync(sn->cpark.p, sim->d_cpark.p, sim->d_cpark.n, cudaMemcpyDeviceToDevice, st));
  }
  PHS_CUDA(sn->pred_cnt.alloc((size_t)sim->total_flows));
  PHS_CUDA(cudaMemcpyAsync(sn->pred_cnt.p, sim->d_pred_cnt.p, sizeof(int32_t) * (size_t)sim->total_flows,
                           cudaMemcpyDeviceToDevice, st));
  sn->res = sim->h_res;
  sn->hist_n = (unsigned long long)sim->h_hist.size();
  if (sim->hist_cap > 0)
    PHS_CUDA(cudaMemcpyAsync(&sn->hist_n, sim->d_hist_n.p, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  sn->cpark_unit_bytes = sim->cpark_unit_bytes;
  sn->cpark_cs = sim->cpark_cs;
  sn->cpark_L = sim->cpark_L;
  sn->cpark_Sc = sim->cpark_Sc;
  sn->n_order = sim->order.size();
  sn->n_cluster = sim->cluster_list.size();
  PHS_CUDA(cudaStreamSynchronize(st));
  sim->snaps.push_back(std::move(sn));
  while ((int)sim->snaps.size() > sim->max_snaps) sim->snaps.pop_front();
  return PHS_OK;
}

// makes snapshot `k` the handle's parked state (and drops the newer ones): the simulation is back at its time
phs_status restore_snapshot(phs_sim *sim, size_t k, cudaStream_t st) {
  phs_sim::Snapshot &sn = *sim->snaps[k];
  if (sn.park.p) PHS_CUDA(cudaMemcpyAsync(sim->d_park.p, sn.park.p, sn.park.n, cudaMemcpyDeviceToDevice, st));
  if (sn.cpark.p) PHS_CUDA(cudaMemcpyAsync(sim->d_cpark.p, sn.cpark.p, sn.cpark.n, cudaMemcpyDeviceToDevice, st));
  PHS_CUDA(cudaMemcpyAsync(sim->d_pred_cnt.p, sn.pred_cnt.p, sizeof(int32_t) * (size_t)sim->total_flows,
                           cudaMemcpyDeviceToDevice, st));
  sim->h_res = sn.res;
  PHS_CUDA(cudaMemcpyAsync(sim->d_res.p, sim->h_res.data(), sizeof(InstResult) * sim->h_res.size(),
                           cudaMemcpyHostToDevice, st));
  if (sim->hist_cap > 0)
    PHS_CUDA(cudaMemcpyAsync(sim->d_hist_n.p, &sn.hist_n, sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
  PHS_CUDA(launch_forget_after(sim->d_tdone.p, sim->d_bneck.p, sim->total_flows, sn.t, st));
  PHS_CUDA(cudaStreamSynchronize(st));
  sim->parked_until = sn.t;
  sim->have_park = true;
  sim->ran = true;
  sim->snaps.resize(k + 1);
  return PHS_OK;
}

// a snapshot is usable while the launch configuration it was parked under still stands
bool snapshot_usable(const phs_sim *sim, const phs_sim::Snapshot &sn) {
  return sn.n_order == sim->order.size() && sn.n_cluster == sim->cluster_list.size() &&
         sn.cpark_unit_bytes == sim->cpark_unit_bytes && sn.cpark_cs == sim->cpark_cs && sn.cpark_L == sim->cpark_L &&
         sn.cpark_Sc == sim->cpark_Sc && (sn.park.n == 0 || sn.park.n == sim->park_stride * sim->units.size()) &&
         (sn.cpark.n == 0 || sn.cpark.n == sim->d_cpark.n);
}

}  // namespace

extern "C" phs_status phs_set_snapshots(phs_sim *sim, int32_t n) {
  PHS_API_BEGIN
  if (!sim || n < 0) return fail(PHS_EINVAL, "bad snapshot count");
  for (auto &c : sim->shards) phs_set_snapshots(c.get(), n);
  sim->max_snaps = n;
  while ((int)sim->snaps.size() > n) sim->snaps.pop_front();
  return PHS_OK;
  PHS_API_END
}

extern "C" phs_status phs_rollback(phs_sim *sim, double t_s) {
  PHS_API_BEGIN
  if (!sim || !(t_s >= 0.0)) return fail(PHS_EINVAL, "bad rollback time");
  for (auto &c : sim->shards) phs_rollback(c.get(), t_s);
  sim->dirty_from = std::min(sim->dirty_from, t_s);
  sim->ran = false;  // no results until the next run
  return PHS_OK;
  PHS_API_END
}

extern "C" phs_status phs_gc(phs_sim *sim, double t_s) {
  PHS_API_BEGIN
  if (!sim || !(t_s >= 0.0)) return fail(PHS_EINVAL, "bad watermark");
  for (auto &c : sim->shards) phs_gc(c.get(), t_s);
  // keep the newest snapshot below the watermark (a rollback to t_s continues from it) and everything later
  while (sim->snaps.size() >= 2 && sim->snaps[1]->t < t_s) sim->snaps.pop_front();
  return PHS_OK;
  PHS_API_END
}

extern "C" phs_status phs_update_flow_start(phs_sim *sim, int32_t instance, int64_t flow, double start) {
  PHS_API_BEGIN
  if (!sim || instance < 0 || instance >= sim->batch) return fail(PHS_EINVAL, "instance out of range");
  if (!(start >= 0.0) || !std::isfinite(start)) return fail(PHS_EINVAL, "start_time_s must be >= 0 and finite");
  Instance &in = sim->inst[(size_t)instance];
  expand_pending(*sim->fab, in);
  if (flow < 0 || flow >= in.n_flows()) return fail(PHS_EINVAL, "flow out of range");
  const double old = in.start[(size_t)flow];
  in.start[(size_t)flow] = start;
  if (!sim->finalized || old == start) return PHS_OK;
  if (!sim->shards.empty()) {  // the shard that holds the instance does the rest, on its device
    const size_t k = (size_t)(std::upper_bound(sim->shard_first.begin(), sim->shard_first.end(), instance) -
                              sim->shard_first.begin()) - 1;
    DeviceGuard guard(sim->devices[k]);
    return phs_update_flow_start(sim->shards[k].get(), instance - sim->shard_first[k], flow, start);
  }
  std::unique_ptr<DeviceGuard> on_device;
  if (sim->devices.size() == 1) on_device.reset(new DeviceGuard(sim->devices[0]));
  const uint32_t p0 = in.pred_off[(size_t)flow], p1 = in.pred_off[(size_t)flow + 1];
  if (p0 == p1) {  // in the sorted initial-activation lists, and in a slot from t = 0: rebuild, start again at 0
    phs_unfinalize(sim);
    return PHS_OK;
  }
  cudaStream_t st = sim->last_stream;
  const int64_t Ft = sim->total_flows;
  if (sim->h_pos.empty()) {  // output position -> position in the per-flow tables (inverse of fmap)
    std::vector<uint32_t> fmap((size_t)Ft);
    PHS_CUDA(cudaMemcpyAsync(fmap.data(), sim->d_fmap.p, sizeof(uint32_t) * (size_t)Ft, cudaMemcpyDeviceToHost, st));
    PHS_CUDA(cudaStreamSynchronize(st));
    sim->h_pos.assign((size_t)Ft, 0);
    for (int64_t p = 0; p < Ft; ++p) sim->h_pos[fmap[(size_t)p]] = (uint32_t)p;
  }
  const int64_t out = sim->flow_base[(size_t)instance] + flow;
  PHS_CUDA(cudaMemcpyAsync(&sim->d_rec.p[sim->h_pos[(size_t)out]].start, &start, sizeof(double), cudaMemcpyHostToDevice, st));
  // release time of the flow in the simulated past = completion of its last predecessor, if all of them are done
  double rel = 0.0;
  bool released = sim->ran || sim->have_park;
  for (uint32_t e = p0; e < p1 && released; ++e) {
    double td = 0.0;
    PHS_CUDA(cudaMemcpyAsync(&td, sim->d_tdone.p + sim->flow_base[(size_t)instance] + in.pred[e], sizeof(double),
                             cudaMemcpyDeviceToHost, st));
    PHS_CUDA(cudaStreamSynchronize(st));
    if (td != td) released = false;
    rel = std::max(rel, td);
  }
  PHS_CUDA(cudaStreamSynchronize(st));
  // from its release on the flow sits in a slot with t_act computed from the old start time: the past is void from
  // there on, unless max(start, release) stays what it was
  if (released && std::max(old, rel) != std::max(start, rel)) {
    sim->dirty_from = std::min(sim->dirty_from, rel);
    sim->ran = false;
  }
  return PHS_OK;
  PHS_API_END
}

extern "C" phs_status phs_run(phs_sim *sim, void *cuda_stream) {
  PHS_API_BEGIN
  return phs_run_until(sim, std::numeric_limits<double>::infinity(), cuda_stream);
  PHS_API_END
}

extern "C" phs_status phs_run_until(phs_sim *sim, double t_stop_s, void *cuda_stream) {
  PHS_API_BEGIN
  if (!sim) return fail(PHS_EINVAL, "null handle");
  if (!(t_stop_s >= 0.0)) return fail(PHS_EINVAL, "t_stop_s must be >= 0");
  if (sim->devices.size() > 1) {  // every device simulates its block of instances, all at once
    if (!sim->finalized) {
      phs_status fs = phs_finalize(sim, nullptr);
      if (fs != PHS_OK) return fs;
    }
    sim->ran = false;
    phs_status rs = for_each_shard(sim, [t_stop_s](size_t, phs_sim *c) { return phs_run_until(c, t_stop_s, nullptr); });
    if (rs != PHS_OK) return rs;
    sim->ran = true;
    return PHS_OK;
  }
  std::unique_ptr<DeviceGuard> on_device;  // phs_set_devices with one device
  if (sim->devices.size() == 1) on_device.reset(new DeviceGuard(sim->devices[0]));
  sim->t_stop = t_stop_s;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (!sim->finalized) {
    phs_status fs = phs_finalize(sim, cuda_stream);
    if (fs != PHS_OK) return fs;
  }
  sim->last_stream = st;
  const int U = (int)sim->units.size();
  PHS_DBG("run: %d units, cta %d cluster %d window %d grid %d", U, (int)sim->order.size(), (int)sim->cluster_list.size(),
          (int)sim->win_list.size(), (int)sim->grid_list.size());
  const bool finite = std::isfinite(sim->t_stop);
  // Resume: a run that stopped at an earlier time left its units parked (shared memory + registers in global
  // memory); a later stop time continues them from there.  When the time goes backwards (or a unit changed its
  // launch configuration after an overflow) the simulation starts again from t = 0 -- it is deterministic, so the
  // results are the same.
  // NEXT-1: if the simulated past is void from dirty_from on (phs_update_flow_start, phs_rollback), or the stop time
  // lies before the parked state, the run continues from the newest snapshot that is early enough -- strictly before
  // dirty_from, not after t_stop -- and only without one from t = 0.
  const double dirty = sim->dirty_from;
  sim->dirty_from = std::numeric_limits<double>::infinity();
  bool resume = sim->have_park && sim->t_stop >= sim->parked_until && sim->parked_until < dirty &&
                (sim->ran || std::isfinite(dirty));
  if (!resume) {
    for (size_t k = sim->snaps.size(); k-- > 0;) {
      const phs_sim::Snapshot &sn = *sim->snaps[k];
      if (!(sn.t < dirty) || !(sn.t <= sim->t_stop) || !snapshot_usable(sim, sn)) continue;
      phs_status rs = restore_snapshot(sim, k, st);
      if (rs != PHS_OK) return rs;
      resume = true;
      break;
    }
    if (!resume) sim->snaps.clear();  // nothing usable: what is left would be later than the state we start from
  }
  sim->resumed_from = resume ? sim->parked_until : 0.0;
  // Until this call succeeds the handle has no results and no parked state: an error return below (history overflow,
  // a unit that does not fit, a CUDA failure) leaves units parked at the NEW stop time, which a later call with an
  // earlier time must not resume from.  Both flags are set again at the end.
  sim->have_park = false;
  sim->ran = false;
  if (finite && !sim->order.empty() && sim->park_stride == 0) {
    sim->park_stride = (sizeof(ParkRegs) + sim->cta.smem + 255) / 256 * 256;
    PHS_CUDA(sim->d_park.alloc(sim->park_stride * (size_t)U));
    PHS_CUDA(cudaMemsetAsync(sim->d_park.p, 0, sim->park_stride * (size_t)U, st));
  }
  DevTables t = tables_of(sim, sim->cta.n_links);
  t.park = (finite || resume) && sim->park_stride ? sim->d_park.p : nullptr;
  t.park_stride = sim->park_stride;
  t.resume = resume ? 1 : 0;
  sim->n_launches = 0;
  sim->resumed_units = 0;
  std::vector<int32_t> cta_list(sim->order), cluster_todo(sim->cluster_list);
  // The window path runs whole simulations only: a stop time, or a resume from parked state, sends its units to the
  // cluster path (same results, one event per iteration).
  const bool use_windows = !finite && !resume;
  sim->win_gang_used = 0;
  if (!use_windows) cluster_todo.insert(cluster_todo.end(), sim->win_list.begin(), sim->win_list.end());
  if (resume) {  // only what has not finished yet
    auto paused = [&](int u) { return sim->h_res[u].status == kPaused; };
    cta_list.erase(std::remove_if(cta_list.begin(), cta_list.end(), [&](int u) { return !paused(u); }), cta_list.end());
    cluster_todo.erase(std::remove_if(cluster_todo.begin(), cluster_todo.end(), [&](int u) { return !paused(u); }),
                       cluster_todo.end());
    if (!cta_list.empty()) PHS_CUDA(sim->d_order2.upload(cta_list, st));
    sim->resumed_units = (int)cta_list.size() + (sim->d_cpark.p ? (int)cluster_todo.size() : 0);
  } else {
    PHS_CUDA(cudaMemsetAsync(sim->d_res.p, 0, sizeof(InstResult) * U, st));  // empty units report status OK
    if (sim->hist_cap > 0) PHS_CUDA(cudaMemsetAsync(sim->d_hist_n.p, 0, sizeof(unsigned long long), st));
    if (finite && sim->total_flows > 0) {  // flows that do not finish by t_stop: NaN / -1
      PHS_CUDA(cudaMemsetAsync(sim->d_tdone.p, 0xff, sizeof(double) * (size_t)sim->total_flows, st));
      PHS_CUDA(cudaMemsetAsync(sim->d_bneck.p, 0xff, sizeof(int32_t) * (size_t)sim->total_flows, st));
    }
  }
  PHS_CUDA(cudaEventRecord(sim->ev0, st));
  if (!cta_list.empty()) {
    sim->n_launches++;
    PHS_CUDA(cudaMemsetAsync(sim->d_ticket.p, 0, sizeof(int), st));
    CtaLaunch cfg = sim->cta;
    cfg.grid = std::min<int>(cfg.grid, (int)cta_list.size());
    PHS_CUDA(launch_cta_path(t, resume ? sim->d_order2.p : sim->d_order.p, (int)cta_list.size(), sim->d_ticket.p, cfg,
                             st));
  }
  PHS_CUDA(cudaEventRecord(sim->ev1, st));
  PHS_CUDA(cudaMemcpyAsync(sim->h_res.data(), sim->d_res.p, sizeof(InstResult) * U, cudaMemcpyDeviceToHost, st));
  PHS_CUDA(cudaStreamSynchronize(st));
  PHS_CUDA(cudaEventElapsedTime(&sim->main_kernel_ms, sim->ev0, sim->ev1));
  // instances that ran out of shared-memory slots on the CTA path move to the cluster path (also for later runs)
  std::vector<int32_t> redo;
  for (int u : cta_list)
    if (sim->h_res[u].status == kOverflow) redo.push_back(u);
  if (!redo.empty()) {
    for (int inst : redo) {
      sim->cluster_list.push_back(inst);
      cluster_todo.push_back(inst);
      sim->order.erase(std::find(sim->order.begin(), sim->order.end(), inst));
    }
    if (!sim->order.empty()) PHS_CUDA(sim->d_order.upload(sim->order, st));
    sim->cta.grid = std::min<int>(sim->cta.grid, std::max<int>(1, (int)sim->order.size()));
    PHS_CUDA(cudaStreamSynchronize(st));
  }
  // window path; units that stop fitting there continue on the cluster path
  if (use_windows && !sim->win_list.empty()) {
    PHS_CUDA(cudaEventRecord(sim->ev0, st));
    std::vector<int32_t> fb;
    phs_status ws = run_window_path(sim, sim->win_list, &fb, st);
    if (ws != PHS_OK) return ws;
    PHS_CUDA(cudaEventRecord(sim->ev1, st));
    PHS_CUDA(cudaStreamSynchronize(st));
    float extra = 0.f;
    PHS_CUDA(cudaEventElapsedTime(&extra, sim->ev0, sim->ev1));
    sim->main_kernel_ms += extra;
    for (int u : fb) {
      sim->cluster_list.push_back(u);
      cluster_todo.push_back(u);
    }
  }
  // cluster path; an instance that overflows a CTA's slot partition is re-run with larger partitions
  std::vector<int32_t> todo(cluster_todo);
  for (int64_t scale = sim->cluster_scale; !todo.empty(); scale *= 2) {
    PHS_CUDA(cudaEventRecord(sim->ev0, st));
    std::vector<int32_t> too_big;
    PHS_DBG("cluster path: %d units, scale %lld", (int)todo.size(), (long long)scale);
    phs_status gs = run_cluster_path(sim, todo, scale, finite, resume, st, &too_big);
    PHS_DBG("cluster path: returned %d, %d too big", (int)gs, (int)too_big.size());
    if (gs != PHS_OK) return gs;
    for (int u : too_big) {  // for good: later runs go straight to the grid path
      sim->grid_list.push_back(u);
      sim->cluster_list.erase(std::remove(sim->cluster_list.begin(), sim->cluster_list.end(), u), sim->cluster_list.end());
      todo.erase(std::remove(todo.begin(), todo.end(), u), todo.end());
    }
    sim->n_launches++;
    PHS_CUDA(cudaEventRecord(sim->ev1, st));
    PHS_CUDA(cudaMemcpyAsync(sim->h_res.data(), sim->d_res.p, sizeof(InstResult) * U, cudaMemcpyDeviceToHost, st));
    PHS_CUDA(cudaStreamSynchronize(st));
    float extra = 0.f;
    PHS_CUDA(cudaEventElapsedTime(&extra, sim->ev0, sim->ev1));
    sim->main_kernel_ms += extra;
    std::vector<int32_t> again;
    for (int i : todo)
      if (sim->h_res[i].status == kOverflow) again.push_back(i);
    if (!again.empty()) {
      if (scale > 64) return fail(PHS_ERANGE, "cluster path: flow slots overflow even at full size");
      sim->cluster_scale = scale * 2;  // remember for later runs
    }
    todo.swap(again);
  }
  // grid path: units that fit no cluster.  They keep no parked state: a later phs_run_until starts them again from
  // t = 0 (deterministic, same results).
  sim->grid_ctas = 0;
  if (!sim->grid_list.empty()) {
    PHS_CUDA(cudaEventRecord(sim->ev0, st));
    phs_status gs = run_grid_path(sim, sim->grid_list, st);
    if (gs != PHS_OK) return gs;
    PHS_CUDA(cudaEventRecord(sim->ev1, st));
    PHS_CUDA(cudaMemcpyAsync(sim->h_res.data(), sim->d_res.p, sizeof(InstResult) * U, cudaMemcpyDeviceToHost, st));
    PHS_CUDA(cudaStreamSynchronize(st));
    float extra = 0.f;
    PHS_CUDA(cudaEventElapsedTime(&extra, sim->ev0, sim->ev1));
    sim->main_kernel_ms += extra;
  }
  if (sim->total_colls > 0) sim->n_launches++;
  PHS_CUDA(launch_collective_times(sim->d_tdone.p, sim->d_coll_first.p, sim->d_coll_n.p, sim->total_colls,
                                   sim->d_coll_t.p, st));
  if (sim->hist_cap > 0) {  // throughput history: fetch, order by (flow, event); a re-run unit repeats its records
    unsigned long long n = 0;
    PHS_CUDA(cudaMemcpyAsync(&n, sim->d_hist_n.p, sizeof(n), cudaMemcpyDeviceToHost, st));
    PHS_CUDA(cudaStreamSynchronize(st));
    if (n > (unsigned long long)sim->hist_cap)
      return fail(PHS_ERANGE, "throughput history needs " + std::to_string(n) + " records, max_records is " +
                                  std::to_string(sim->hist_cap));
    sim->h_hist.resize((size_t)n);
    if (n) PHS_CUDA(cudaMemcpyAsync(sim->h_hist.data(), sim->d_hist.p, sizeof(HistRec) * n, cudaMemcpyDeviceToHost, st));
    PHS_CUDA(cudaStreamSynchronize(st));
    std::sort(sim->h_hist.begin(), sim->h_hist.end(), [](const HistRec &a, const HistRec &b) {
      return a.flow != b.flow ? a.flow < b.flow : a.ev < b.ev;
    });
    sim->h_hist.erase(std::unique(sim->h_hist.begin(), sim->h_hist.end(),
                                  [](const HistRec &a, const HistRec &b) { return a.flow == b.flow && a.ev == b.ev; }),
                      sim->h_hist.end());
  }
  sim->ran = true;
  sim->have_park = finite;
  sim->parked_until = sim->t_stop;
  if (finite) {
    phs_status ss = take_snapshot(sim, st);
    if (ss != PHS_OK) return ss;
  }
  for (int u = 0; u < U; ++u) {
    const int i = sim->units[u].inst;
    if (sim->h_res[u].status == PHS_ECYCLE)
      return fail(PHS_ECYCLE, "instance " + std::to_string(i) + ": flows left waiting on dependencies that never complete");
    if (sim->h_res[u].status != PHS_OK && sim->h_res[u].status != kPaused)
      return fail(PHS_ECUDA, "instance " + std::to_string(i) + ": unexpected kernel status " +
                                 std::to_string(sim->h_res[u].status));
  }
  return PHS_OK;
  PHS_API_END
}


// phs_run without allocation (include/phs.h): every unit on the grid path, the kernel's scratch in the library's static
// __device__ array (phs_grid.cu).  Only enqueues kernels, memsets and copies on buffers phs_finalize made.
extern "C" phs_status phs_run_static(phs_sim *sim, void *cuda_stream, double *t_done_dev, int32_t *bneck_dev, int64_t n) {
  PHS_API_BEGIN
  if (!sim) return fail(PHS_EINVAL, "null handle");
  if (!sim->shards.empty() || sim->devices.size() > 1)
    return fail(PHS_ESTATE, "phs_run_static: the handle is bound to several devices");
  if (!sim->finalized) return fail(PHS_ESTATE, "phs_run_static builds nothing: call phs_finalize first");
  if (sim->want_log || sim->hist_cap > 0)
    return fail(PHS_ESTATE, "phs_run_static: the grid path writes no event log and the static run keeps no history");
  if (n != sim->total_flows) return fail(PHS_EINVAL, "n must equal the total flow count");
  const int U = (int)sim->units.size();
  int64_t Fm = 1;
  int Lm = 1;
  for (int u = 0; u < U; ++u) {
    Fm = std::max<int64_t>(Fm, sim->units[(size_t)u].n_flows);
    Lm = std::max(Lm, sim->units[(size_t)u].n_links);
  }
  if (U > PHS_STATIC_MAX_UNITS)
    return fail(PHS_ERANGE, "phs_run_static: " + std::to_string(U) + " simulation units, the static unit list holds " +
                                std::to_string(PHS_STATIC_MAX_UNITS));
  if (grid_scratch_bytes(Fm, Lm) > grid_static_capacity())
    return fail(PHS_ERANGE, "phs_run_static: the largest unit (" + std::to_string(Fm) + " flows, " + std::to_string(Lm) +
                                " links) needs " + std::to_string(grid_scratch_bytes(Fm, Lm)) +
                                " bytes of state, the static scratch holds " + std::to_string(grid_static_capacity()));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int cur = 0;
  PHS_CUDA(cudaGetDevice(&cur));
  const int want = sim->devices.size() == 1 ? sim->devices[0] : cur;
  struct Restore {  // phs_set_devices with one device: run there, leave the caller's device as it was
    int dev;
    bool on;
    ~Restore() {
      if (on) cudaSetDevice(dev);
    }
  } restore{cur, want != cur};
  if (want != cur) PHS_CUDA(cudaSetDevice(want));
  // like phs_run: until the call succeeds the handle has no results and no parked state
  // (dirty_from is left alone: snapshots later than it stay void for the next phs_run_until)
  sim->t_stop = std::numeric_limits<double>::infinity();
  sim->have_park = false;
  sim->ran = false;
  sim->last_stream = st;
  sim->resumed_from = 0.0;
  sim->resumed_units = 0;
  sim->win_gang_used = 0;
  sim->n_launches = 0;
  sim->grid_ctas = 0;
  sim->main_kernel_ms = 0.f;
  if (U > 0) {
    int n_ctas = 0;
    PHS_CUDA(grid_max_ctas(&n_ctas));
    if (n_ctas < 1) return fail(PHS_ECUDA, "grid path: the kernel cannot be resident");
    n_ctas = (int)std::max<int64_t>(1, std::min<int64_t>(n_ctas, (Fm + kGridThreads - 1) / kGridThreads));
    PHS_CUDA(cudaMemsetAsync(sim->d_res.p, 0, sizeof(InstResult) * (size_t)U, st));  // empty units report status OK
    PHS_CUDA(cudaEventRecord(sim->ev0, st));
    PHS_CUDA(launch_grid_static(tables_of(sim, Lm), U, Fm, Lm, n_ctas, st));
    PHS_CUDA(cudaEventRecord(sim->ev1, st));
    sim->grid_ctas = n_ctas;
    sim->n_launches = 2;  // the unit-list kernel and the grid kernel
    PHS_CUDA(cudaMemcpyAsync(sim->h_res.data(), sim->d_res.p, sizeof(InstResult) * (size_t)U, cudaMemcpyDeviceToHost, st));
  }
  if (sim->total_colls > 0) sim->n_launches++;
  PHS_CUDA(launch_collective_times(sim->d_tdone.p, sim->d_coll_first.p, sim->d_coll_n.p, sim->total_colls,
                                   sim->d_coll_t.p, st));
  if (t_done_dev && n > 0)
    PHS_CUDA(cudaMemcpyAsync(t_done_dev, sim->d_tdone.p, sizeof(double) * (size_t)n, cudaMemcpyDeviceToDevice, st));
  if (bneck_dev && n > 0)
    PHS_CUDA(cudaMemcpyAsync(bneck_dev, sim->d_bneck.p, sizeof(int32_t) * (size_t)n, cudaMemcpyDeviceToDevice, st));
  PHS_CUDA(cudaStreamSynchronize(st));
  if (U > 0) PHS_CUDA(cudaEventElapsedTime(&sim->main_kernel_ms, sim->ev0, sim->ev1));
  sim->ran = true;
  sim->parked_until = sim->t_stop;
  for (int u = 0; u < U; ++u) {
    const int i = sim->units[(size_t)u].inst;
    if (sim->h_res[(size_t)u].status == PHS_ECYCLE)
      return fail(PHS_ECYCLE, "instance " + std::to_string(i) + ": flows left waiting on dependencies that never complete");
    if (sim->h_res[(size_t)u].status != PHS_OK)
      return fail(PHS_ECUDA, "instance " + std::to_string(i) + ": unexpected kernel status " +
                                 std::to_string(sim->h_res[(size_t)u].status));
  }
  return PHS_OK;
  PHS_API_END
}
