// phs_build.cpp -- host builder: link numbering, seeded ECMP routing (flow -> link CSR incidence) and the
// collective -> flow decomposer with its dependency DAG.  Pure host C++, no CUDA.  DESIGN.md S1-S3; the
// passages of the paper are PAPER.md L98 (topology, multipath routing) and L104 (ring all-reduce, flows with
// timestamps).
#include <algorithm>
#include <cmath>
#include <limits>

#include "phs_internal.h"

namespace phs {

// ------------------------------------------------------------------------------------------------ Fabric (S1)
// Directed link ids, in blocks:
//   [0, 2G)            NVLink : 2g GPU->NVSwitch, 2g+1 NVSwitch->GPU
//   [2G, 4G)           NIC    : 2G+2g GPU->tier-1 switch, 2G+2g+1 back
//   [tier1_base, ...)  tier1<->tier2 pairs u: up tier1_base+2u, down tier1_base+2u+1
//   [tier2_base, ...)  fat tree tier2<->tier3 pairs
phs_status Fabric::validate(const phs_topology_desc &d, std::string *why) {
  auto bad = [&](const char *m) {
    if (why) *why = m;
    return PHS_EINVAL;
  };
  auto cap_ok = [](double c) { return c > 0.0 && c < 0x1p42; };
  if (d.n_hosts <= 0 || d.gpus_per_host <= 0) return bad("n_hosts and gpus_per_host must be positive");
  if (!cap_ok(d.nvlink_Bps) || !cap_ok(d.nic_Bps)) return bad("nvlink_Bps / nic_Bps must be in (0, 2^42)");
  if (!(d.hop_latency_s >= 0.0) || !std::isfinite(d.hop_latency_s)) return bad("hop_latency_s must be >= 0");
  int64_t links = 4LL * d.n_hosts * d.gpus_per_host;
  switch (d.kind) {
    case PHS_TOPO_SINGLE:
      break;
    case PHS_TOPO_LEAF_SPINE:
      if (d.n_leaves <= 0 || d.n_spines <= 0 || d.uplinks_per_leaf_spine <= 0)
        return bad("leaf-spine needs n_leaves, n_spines, uplinks_per_leaf_spine > 0");
      if (d.n_hosts % d.n_leaves) return bad("n_hosts must be a multiple of n_leaves");
      if (!cap_ok(d.fabric_Bps)) return bad("fabric_Bps must be in (0, 2^42)");
      links += 2LL * d.n_leaves * d.n_spines * d.uplinks_per_leaf_spine;
      break;
    case PHS_TOPO_FAT_TREE:
      if (d.k < 2 || (d.k & 1) || d.agg_uplinks <= 0) return bad("fat tree needs even k >= 2 and agg_uplinks > 0");
      if (d.gpus_per_host != d.k / 2 || d.n_hosts != d.k * (d.k / 2))
        return bad("fat tree needs gpus_per_host = k/2 and n_hosts = k*k/2");
      if (!cap_ok(d.fabric_Bps)) return bad("fabric_Bps must be in (0, 2^42)");
      links += 2LL * d.k * (d.k / 2) * (d.k / 2) + 2LL * d.k * (d.k / 2) * d.agg_uplinks;
      break;
    default:
      return bad("unknown topology kind");
  }
  if (d.compute_lanes < 0 || d.compute_lanes > 64) return bad("compute_lanes must be in [0, 64]");
  links += (int64_t)d.n_hosts * d.gpus_per_host * d.compute_lanes;
  if (links > 0x3fffffff) {
    if (why) *why = "too many links";
    return PHS_ERANGE;
  }
  return PHS_OK;
}

Fabric::Fabric(const phs_topology_desc &d) : d_(d) {
  gpus_ = d.n_hosts * d.gpus_per_host;
  tier1_base_ = 4 * gpus_;
  tier2_base_ = tier1_base_;
  links_ = tier1_base_;
  if (d.kind == PHS_TOPO_LEAF_SPINE) {
    links_ += 2 * d.n_leaves * d.n_spines * d.uplinks_per_leaf_spine;
  } else if (d.kind == PHS_TOPO_FAT_TREE) {
    const int half = d.k / 2;
    tier2_base_ = tier1_base_ + 2 * d.k * half * half;
    links_ = tier2_base_ + 2 * d.k * half * d.agg_uplinks;
  }
  net_links_ = links_;
  links_ += gpus_ * d.compute_lanes;  // compute engine links (phs_add_spans) follow the network links
}

// ------------------------------------------------------------------------------------------------ graph (S8)
phs_status Fabric::validate_graph(const GraphLinks &g, std::string *why) {
  auto bad = [&](const char *m) {
    if (why) *why = m;
    return PHS_EINVAL;
  };
  if (g.n_gpus < 2 || g.n_nodes < g.n_gpus) return bad("a graph topology needs n_gpus >= 2 and n_nodes >= n_gpus");
  if (g.compute_lanes < 0 || g.compute_lanes > 64) return bad("compute_lanes must be in [0, 64]");
  if (g.from.empty()) return bad("a graph topology needs links");
  for (size_t i = 0; i < g.from.size(); ++i) {
    if (g.from[i] < 0 || g.from[i] >= g.n_nodes || g.to[i] < 0 || g.to[i] >= g.n_nodes || g.from[i] == g.to[i])
      return bad("link endpoint out of range");
    if (!(g.cap[i] > 0.0) || !(g.cap[i] < 0x1p42)) return bad("link capacity must be in (0, 2^42) byte/s");
    if (!(g.lat[i] >= 0.0) || !std::isfinite(g.lat[i])) return bad("link latency must be >= 0 and finite");
  }
  if ((int64_t)g.from.size() + (int64_t)g.n_gpus * g.compute_lanes > 0x3fffffff) {
    if (why) *why = "too many links";
    return PHS_ERANGE;
  }
  return PHS_OK;
}

Fabric::Fabric(GraphLinks g) : d_{}, graph_(true), g_(std::move(g)) {
  d_.kind = 3;
  d_.n_hosts = g_.n_gpus;
  d_.gpus_per_host = 1;
  d_.compute_lanes = g_.compute_lanes;
  gpus_ = g_.n_gpus;
  net_links_ = (int32_t)g_.from.size();
  links_ = net_links_ + gpus_ * g_.compute_lanes;
  tier1_base_ = tier2_base_ = net_links_;
  const int N = g_.n_nodes;
  // out-links grouped by node: link ids sorted by (from, id)
  out_link_.resize((size_t)net_links_);
  for (int32_t i = 0; i < net_links_; ++i) out_link_[(size_t)i] = i;
  std::stable_sort(out_link_.begin(), out_link_.end(), [&](int32_t a, int32_t b) { return g_.from[a] < g_.from[b]; });
  out_off_.assign((size_t)N + 1, 0);
  for (int32_t i = 0; i < net_links_; ++i) out_off_[(size_t)g_.from[i] + 1]++;
  for (int v = 0; v < N; ++v) out_off_[(size_t)v + 1] += out_off_[(size_t)v];
  // hop distance of every node to every GPU: level-synchronous search over the in-links
  std::vector<std::vector<int32_t>> in_links((size_t)N);
  for (int32_t i = 0; i < net_links_; ++i) in_links[(size_t)g_.to[i]].push_back(i);
  hops_.assign((size_t)gpus_ * N, -1);
  std::vector<int32_t> frontier, next;
  for (int g0 = 0; g0 < gpus_; ++g0) {
    int16_t *h = hops_.data() + (size_t)g0 * N;
    h[g0] = 0;
    frontier.assign(1, g0);
    for (int16_t level = 1; !frontier.empty(); ++level) {
      next.clear();
      for (int32_t v : frontier)
        for (int32_t l : in_links[(size_t)v]) {
          const int32_t u = g_.from[(size_t)l];
          if (h[u] < 0) {
            h[u] = level;
            next.push_back(u);
          }
        }
      frontier.swap(next);
    }
  }
}

bool Fabric::routable(int32_t src, int32_t dst) const {
  if (!graph_ || src == dst) return true;
  const int16_t h = hops_[(size_t)dst * g_.n_nodes + src];
  return h >= 1 && h <= kMaxHops;
}

double Fabric::default_capacity(int32_t link) const {
  if (link >= net_links_) return 0x1p32;  // work units per second of a compute lane
  if (graph_) return g_.cap[(size_t)link];
  if (link < 2 * gpus_) return d_.nvlink_Bps;
  if (link < 4 * gpus_) return d_.nic_Bps;
  if (link >= net_links_) return 0x1p32;  // work units per second of a compute lane
  return d_.fabric_Bps;
}

// SplitMix64 step: add the golden-gamma constant, then the xor-shift-multiply finaliser.
uint64_t splitmix64_step(uint64_t x) {
  x += 0x9E3779B97F4A7C15ULL;
  x ^= x >> 30;
  x *= 0xBF58476D1CE4E5B9ULL;
  x ^= x >> 27;
  x *= 0x94D049BB133111EBULL;
  x ^= x >> 31;
  return x;
}

// ------------------------------------------------------------------------------------------------ ECMP (S2)
int Fabric::route(uint64_t seed, int32_t src, int32_t dst, int32_t conn, int32_t *out) const {
  if (src == dst) {  // a compute span: the engine link of lane `conn` of the GPU
    out[0] = net_links_ + src * d_.compute_lanes + conn;
    return 1;
  }
  if (graph_) {  // S8: walk towards dst along shortest paths; hop k takes candidate mix(H ^ (k+1)) mod #candidates
    uint64_t h = splitmix64_step(seed);
    h = splitmix64_step(h ^ (uint64_t)(uint32_t)src);
    h = splitmix64_step(h ^ (uint64_t)(uint32_t)dst);
    h = splitmix64_step(h ^ (uint64_t)(uint32_t)conn);
    const int16_t *left = hops_.data() + (size_t)dst * g_.n_nodes;
    int n = 0;
    for (int32_t at = src; at != dst && n < kMaxHops;) {
      const uint64_t pick = splitmix64_step(h ^ (uint64_t)(n + 1));
      // count the candidates, then take the pick-th (out-links are in ascending link id)
      int n_cand = 0;
      for (int32_t e = out_off_[(size_t)at]; e < out_off_[(size_t)at + 1]; ++e)
        n_cand += left[g_.to[(size_t)out_link_[(size_t)e]]] == left[at] - 1;
      int want = (int)(pick % (uint64_t)n_cand);
      for (int32_t e = out_off_[(size_t)at]; e < out_off_[(size_t)at + 1]; ++e) {
        const int32_t l = out_link_[(size_t)e];
        if (left[g_.to[(size_t)l]] != left[at] - 1) continue;
        if (want-- == 0) {
          out[n++] = l;
          at = g_.to[(size_t)l];
          break;
        }
      }
    }
    return n;
  }
  const int gph = d_.gpus_per_host;
  const int host_s = src / gph, host_d = dst / gph;
  if (host_s == host_d) {  // stays on the host's NVSwitch
    out[0] = 2 * src;
    out[1] = 2 * dst + 1;
    return 2;
  }
  const int32_t first = 2 * gpus_ + 2 * src, last = 2 * gpus_ + 2 * dst + 1;
  int n = 0;
  out[n++] = first;
  if (d_.kind != PHS_TOPO_SINGLE) {
    uint64_t h = splitmix64_step(seed);
    h = splitmix64_step(h ^ (uint64_t)(uint32_t)src);
    h = splitmix64_step(h ^ (uint64_t)(uint32_t)dst);
    h = splitmix64_step(h ^ (uint64_t)(uint32_t)conn);
    const uint32_t hi_word = (uint32_t)(h >> 32);
    if (d_.kind == PHS_TOPO_LEAF_SPINE) {
      const int hosts_per_leaf = d_.n_hosts / d_.n_leaves;
      const int leaf_s = host_s / hosts_per_leaf, leaf_d = host_d / hosts_per_leaf;
      if (leaf_s != leaf_d) {
        const int P = d_.uplinks_per_leaf_spine;
        const int choice = (int)(h % (uint64_t)(d_.n_spines * P));
        const int spine = choice / P, lane_up = choice % P, lane_dn = (int)((uint64_t)hi_word % (uint64_t)P);
        out[n++] = tier1_base_ + 2 * ((leaf_s * d_.n_spines + spine) * P + lane_up);
        out[n++] = tier1_base_ + 2 * ((leaf_d * d_.n_spines + spine) * P + lane_dn) + 1;
      }
    } else {  // fat tree: a host hangs off its own edge switch
      const int half = d_.k / 2;
      const int pod_s = host_s / half, edge_s = host_s % half, pod_d = host_d / half, edge_d = host_d % half;
      const int agg = (int)(h % (uint64_t)half);
      const int up1 = tier1_base_ + 2 * ((pod_s * half + edge_s) * half + agg);
      const int dn1 = tier1_base_ + 2 * ((pod_d * half + edge_d) * half + agg) + 1;
      out[n++] = up1;
      if (pod_s != pod_d) {
        const int U = d_.agg_uplinks;
        const int core_lane = (int)((uint64_t)hi_word % (uint64_t)U);
        out[n++] = tier2_base_ + 2 * ((pod_s * half + agg) * U + core_lane);
        out[n++] = tier2_base_ + 2 * ((pod_d * half + agg) * U + core_lane) + 1;
      }
      out[n++] = dn1;
    }
  }
  out[n++] = last;
  return n;
}

// ------------------------------------------------------------------------------------------------ flows
namespace {

// Adds one flow (without dependencies) and returns its id.
int32_t push_flow(const Fabric &fab, Instance &inst, int32_t src, int32_t dst, double bytes, double start,
                  int32_t conn) {
  int32_t hops[kMaxHops];
  const int n = fab.route(inst.seed, src, dst, conn, hops);
  double lat = 0.0;
  for (int i = 0; i < n; ++i) {
    inst.path.push_back(hops[i]);
    lat = lat + fab.latency(hops[i]);
  }
  inst.src.push_back(src);
  inst.dst.push_back(dst);
  inst.bytes.push_back(bytes);
  inst.start.push_back(start);
  inst.lat.push_back(lat);
  inst.path_off.push_back((uint32_t)inst.path.size());
  inst.pred_off.push_back((uint32_t)inst.pred.size());
  return (int32_t)inst.src.size() - 1;
}

// Adds a copy of flow `of` that starts at 0 and has no dependencies yet: same endpoints, bytes, path and latency.
void repeat_flow(Instance &inst, size_t of) {
  int32_t hops[kMaxHops];
  const uint32_t p0 = inst.path_off[of], n = inst.path_off[of + 1] - p0;
  for (uint32_t h = 0; h < n; ++h) hops[h] = inst.path[p0 + h];
  inst.path.insert(inst.path.end(), hops, hops + n);
  inst.src.push_back(inst.src[of]);
  inst.dst.push_back(inst.dst[of]);
  inst.bytes.push_back(inst.bytes[of]);
  inst.start.push_back(0.0);
  inst.lat.push_back(inst.lat[of]);
  inst.path_off.push_back((uint32_t)inst.path.size());
  inst.pred_off.push_back((uint32_t)inst.pred.size());
}

// A dependency of the flow pushed last.
inline void push_dep(Instance &inst, int32_t on) {
  inst.pred.push_back(on);
  inst.pred_off.back() = (uint32_t)inst.pred.size();
}

// Flows of collective `a` that must finish before rank `rho` may start a later collective: what rho sent and
// what rho received in a's last step (ring), everything from / to rho (all-to-all), or what rho sends and receives
// in a's last chunk (chain and tree kinds; positions worked out from the decomposition rule, see expand_collective).
void chain_after(Instance &inst, const Collective &a, int32_t rho) {
  int pos = -1;
  for (int i = 0; i < a.n_ranks; ++i)
    if (a.ranks[i] == rho) {
      pos = i;
      break;
    }
  if (pos < 0) return;  // rho did not take part: no edge
  const int N = a.n_ranks;
  if (a.kind == PHS_ALLTOALL) {
    for (int other = 0; other < N; ++other) {
      if (other == pos) continue;
      push_dep(inst, a.first_flow + pos * (N - 1) + (other > pos ? other - 1 : other));  // pos -> other
      push_dep(inst, a.first_flow + other * (N - 1) + (pos > other ? pos - 1 : pos));    // other -> pos
    }
  } else if (a.kind == PHS_BROADCAST_CHAIN || a.kind == PHS_REDUCE_CHAIN) {
    // hop i of the last chunk: broadcast r[i] -> r[i+1]; reduce r[N-1-i] -> r[N-2-i].  In ascending flow id.
    const int32_t last = a.first_flow + (a.chunks - 1) * (N - 1);
    const int q = a.kind == PHS_BROADCAST_CHAIN ? pos : N - 1 - pos;  // rho sends hop q and receives hop q-1
    if (q >= 1) push_dep(inst, last + q - 1);
    if (q <= N - 2) push_dep(inst, last + q);
  } else if (a.kind == PHS_ALLREDUCE_TREE) {
    // last chunk's block: up(i) at offset i-1, down(i) at offset (N-1) + i-1.  rho at position pos sends up(pos) and
    // down(children), receives up(children) and down(pos).  In ascending flow id.
    const int32_t blk = a.first_flow + (a.chunks - 1) * 2 * (N - 1);
    const int l = 2 * pos + 1, r = 2 * pos + 2;
    if (pos >= 1) push_dep(inst, blk + pos - 1);
    if (l < N) push_dep(inst, blk + l - 1);
    if (r < N) push_dep(inst, blk + r - 1);
    if (pos >= 1) push_dep(inst, blk + (N - 1) + pos - 1);
    if (l < N) push_dep(inst, blk + (N - 1) + l - 1);
    if (r < N) push_dep(inst, blk + (N - 1) + r - 1);
  } else {
    const int32_t last_step = a.first_flow + (a.steps - 1) * a.n_ranks;
    push_dep(inst, last_step + pos);                                  // sent by rho
    push_dep(inst, last_step + (pos == 0 ? a.n_ranks - 1 : pos - 1));  // received by rho
  }
}

}  // namespace

phs_status append_collective(const Fabric &fab, Instance &inst, int32_t kind, const int32_t *ranks, int32_t N,
                             double bytes, double start, const int32_t *after, int32_t n_after,
                             const int64_t *after_flows, int32_t n_after_flows, int32_t chunks, std::string *why,
                             bool checked) {
  auto bad = [&](const char *m) {
    if (why) *why = m;
    return PHS_EINVAL;
  };
  // `checked`: the same kind / ranks / after lists were validated on another instance of the same topology with as many
  // collectives (phs_add_collective_batch); only what depends on the instance is looked at again
  if (checked) goto record;
  if (!ranks) return bad("ranks is null");
  if (kind < PHS_ALLREDUCE_RING || kind > PHS_ALLREDUCE_TREE) return bad("unknown collective kind");
  if (chunks < 1 || chunks > 65536) return bad("chunks must be in [1, 65536]");
  if (kind <= PHS_ALLTOALL && chunks != 1) return bad("chunks applies to the chain and tree kinds only");
  if (N < 2) return bad("a collective needs at least 2 ranks");
  if (!(bytes > 0.0) || !std::isfinite(bytes)) return bad("bytes must be positive and finite");
  if (!(start >= 0.0) || !std::isfinite(start)) return bad("start_time_s must be >= 0 and finite");
  if (n_after < 0 || (n_after > 0 && !after)) return bad("bad after_coll_ids");
  {
    std::vector<uint8_t> seen((size_t)fab.n_gpus(), 0);
    for (int i = 0; i < N; ++i) {
      if (ranks[i] < 0 || ranks[i] >= fab.n_gpus()) return bad("rank out of range");
      if (seen[ranks[i]]) return bad("duplicate rank in collective");
      seen[ranks[i]] = 1;
    }
  }
  for (int a = 0; a < n_after; ++a)
    if (after[a] < 0 || after[a] >= (int32_t)inst.colls.size()) return bad("after_coll_ids names an unknown collective");
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j)
      if (!fab.routable(ranks[i], ranks[j])) return bad("two ranks of the collective have no route of at most 6 links");
  if (n_after_flows < 0 || (n_after_flows > 0 && !after_flows)) return bad("bad after_flow_ids");
  for (int a = 0; a < n_after_flows; ++a)
    if (after_flows[a] < 0 || after_flows[a] >= inst.n_flows()) return bad("after_flow_ids must name earlier flows");
record:
  const int steps = kind == PHS_ALLREDUCE_RING ? 2 * (N - 1) : kind == PHS_ALLTOALL ? 1 : N - 1;
  const int64_t nf = kind == PHS_ALLTOALL          ? (int64_t)N * (N - 1)
                     : kind == PHS_ALLREDUCE_TREE  ? (int64_t)chunks * 2 * (N - 1)
                     : kind >= PHS_BROADCAST_CHAIN ? (int64_t)chunks * (N - 1)
                                                   : (int64_t)steps * N;
  if (inst.n_flows() + nf > 0x7ffffff0LL) {
    if (why) *why = "too many flows in one instance";
    return PHS_ERANGE;
  }
  Collective c;
  c.kind = kind;
  c.n_ranks = N;
  c.first_flow = (int32_t)inst.n_flows();
  c.n_flows = (int32_t)nf;
  c.steps = steps;
  c.chunks = chunks;
  c.ranks.assign(ranks, ranks + N);
  c.chain = (int32_t)inst.colls.size();
  for (int a = 0; a < n_after; ++a) c.chain = std::min(c.chain, inst.colls[after[a]].chain);
  c.bytes = bytes;
  c.start = start;
  c.after.assign(after, after + n_after);
  c.after_flows.assign(after_flows, after_flows + n_after_flows);
  inst.flow_count += nf;
  inst.colls.push_back(std::move(c));
  return PHS_OK;
}

namespace {

// S3: the flows and dependencies of collective `id`, appended at flow id first_flow.
void expand_collective(const Fabric &fab, Instance &inst, int32_t id) {
  const Collective &c = inst.colls[(size_t)id];
  const int N = c.n_ranks, steps = c.steps;
  const int32_t *ranks = c.ranks.data();
  const int32_t *after = c.after.data();
  const int n_after = (int)c.after.size();
  const double start = c.start;
  const int32_t conn = id;  // ECMP key: one path per (pair, collective)
  // dependencies of an initial flow sent by rank rho: the `after` collectives, then the listed earlier flows / spans
  // that start or end at rho
  auto initial_edges = [&](int32_t rho) {
    for (int k = 0; k < n_after; ++k) chain_after(inst, inst.colls[after[k]], rho);
    for (int32_t f : inst.colls[(size_t)id].after_flows)
      if (inst.src[(size_t)f] == rho || inst.dst[(size_t)f] == rho) push_dep(inst, f);
  };
  const double chunk = c.bytes / (double)N;
  if (c.kind == PHS_BROADCAST_CHAIN || c.kind == PHS_REDUCE_CHAIN) {
    // NEXT-3: pipelined chain.  Hop i carries every chunk in turn: chunk-major flow order, hop i of
    // chunk ch waits for hop i-1 of the same chunk (the data is there) and for hop i of the previous chunk (FIFO).
    // Chunks ch > 0 take the route of chunk 0 (ECMP keys on pair + collective).
    const double piece = c.bytes / (double)c.chunks;
    const int hops = N - 1;
    for (int ch = 0; ch < c.chunks; ++ch)
      for (int i = 0; i < hops; ++i) {
        if (ch == 0) {
          const int a = c.kind == PHS_BROADCAST_CHAIN ? i : N - 1 - i, b = c.kind == PHS_BROADCAST_CHAIN ? i + 1 : N - 2 - i;
          push_flow(fab, inst, ranks[a], ranks[b], piece, i == 0 ? start : 0.0, conn);
          if (i == 0) initial_edges(ranks[a]);
        } else {
          repeat_flow(inst, (size_t)c.first_flow + (size_t)i);
        }
        if (i > 0) push_dep(inst, c.first_flow + ch * hops + i - 1);
        if (ch > 0) push_dep(inst, c.first_flow + (ch - 1) * hops + i);
      }
  } else if (c.kind == PHS_ALLREDUCE_TREE) {
    // NEXT-3: binary tree in heap order; per chunk the N-1 up flows (child -> parent), then the N-1 down flows
    const double piece = c.bytes / (double)c.chunks;
    const int blk = 2 * (N - 1);
    for (int ch = 0; ch < c.chunks; ++ch) {
      const int32_t base = c.first_flow + ch * blk, prev = base - blk;
      for (int i = 1; i < N; ++i) {  // up(ch, i)
        const int l = 2 * i + 1, r = 2 * i + 2;
        const bool leaf_first = ch == 0 && l >= N;
        if (ch == 0) {
          push_flow(fab, inst, ranks[i], ranks[(i - 1) / 2], piece, leaf_first ? start : 0.0, conn);
          if (leaf_first) initial_edges(ranks[i]);
        } else {
          repeat_flow(inst, (size_t)c.first_flow + (size_t)(i - 1));
        }
        if (l < N) push_dep(inst, base + l - 1);
        if (r < N) push_dep(inst, base + r - 1);
        if (ch > 0) push_dep(inst, prev + i - 1);
      }
      for (int i = 1; i < N; ++i) {  // down(ch, i)
        const int p = (i - 1) / 2;
        if (ch == 0)
          push_flow(fab, inst, ranks[p], ranks[i], piece, 0.0, conn);
        else
          repeat_flow(inst, (size_t)c.first_flow + (size_t)(N - 1 + i - 1));
        if (p == 0) {  // the root has the chunk's sum once both of its children have delivered
          push_dep(inst, base + 0);
          if (N > 2) push_dep(inst, base + 1);
        } else {
          push_dep(inst, base + (N - 1) + p - 1);
        }
        if (ch > 0) push_dep(inst, prev + (N - 1) + i - 1);
      }
    }
  } else if (c.kind == PHS_ALLTOALL) {
    for (int i = 0; i < N; ++i)
      for (int j = 0; j < N; ++j) {
        if (i == j) continue;
        push_flow(fab, inst, ranks[i], ranks[j], chunk, start, conn);
        initial_edges(ranks[i]);
      }
  } else {
    // step-major: flow (s, i) sends chunk from ranks[i] to ranks[i+1]; it waits for the chunk it forwards
    // (s-1, i-1) and for the sender's previous send (s-1, i) -- FIFO per connection.  ECMP keys on (pair,
    // collective), so step s > 0 of ring position i takes the path of step 0 and copies it.
    for (int s = 0; s < steps; ++s) {
      const int32_t prev = c.first_flow + (s - 1) * N;
      for (int i = 0; i < N; ++i) {
        if (s == 0) {
          const int next_rank = i + 1 == N ? 0 : i + 1;
          push_flow(fab, inst, ranks[i], ranks[next_rank], chunk, start, conn);
          initial_edges(ranks[i]);
        } else {
          repeat_flow(inst, (size_t)c.first_flow + (size_t)i);
          push_dep(inst, prev + (i == 0 ? N - 1 : i - 1));
          push_dep(inst, prev + i);
        }
      }
    }
  }
}

}  // namespace

void expand_pending(const Fabric &fab, Instance &inst) {
  if (inst.expanded == inst.colls.size()) return;
  const size_t F = (size_t)inst.flow_count;
  inst.src.reserve(F);
  inst.dst.reserve(F);
  inst.bytes.reserve(F);
  inst.start.reserve(F);
  inst.lat.reserve(F);
  inst.path_off.reserve(F + 1);
  inst.pred_off.reserve(F + 1);
  for (; inst.expanded < inst.colls.size(); ++inst.expanded) expand_collective(fab, inst, (int32_t)inst.expanded);
}

phs_status append_flows(const Fabric &fab, Instance &inst, int64_t n, const int32_t *src, const int32_t *dst,
                        const double *bytes, const double *start, const int64_t *dep_off, const int64_t *dep_ids,
                        const int32_t *conn_id, std::string *why) {
  auto bad = [&](const char *m) {
    if (why) *why = m;
    return PHS_EINVAL;
  };
  if (n < 0 || (n > 0 && (!src || !dst || !bytes))) return bad("null flow arrays");
  expand_pending(fab, inst);  // flow ids follow submission order
  const int64_t first = inst.n_flows();
  if (first + n > 0x7ffffff0LL) {
    if (why) *why = "too many flows in one instance";
    return PHS_ERANGE;
  }
  for (int64_t i = 0; i < n; ++i) {  // validate first, mutate after
    if (src[i] < 0 || src[i] >= fab.n_gpus() || dst[i] < 0 || dst[i] >= fab.n_gpus()) return bad("rank out of range");
    if (src[i] == dst[i]) return bad("src == dst");
    if (!fab.routable(src[i], dst[i])) return bad("no route of at most 6 links between src and dst");
    if (!(bytes[i] > 0.0) || !std::isfinite(bytes[i])) return bad("bytes must be positive and finite");
    if (start && (!(start[i] >= 0.0) || !std::isfinite(start[i]))) return bad("start_time_s must be >= 0 and finite");
    if (dep_off) {
      if (dep_off[i + 1] < dep_off[i]) return bad("dep_off must be non-decreasing");
      if (dep_off[i + 1] > dep_off[i] && !dep_ids) return bad("dep_flow_ids is null");
      for (int64_t e = dep_off[i]; e < dep_off[i + 1]; ++e)
        if (dep_ids[e] < 0 || dep_ids[e] >= first + i) return bad("a flow may only depend on earlier flows");
    }
  }
  for (int64_t i = 0; i < n; ++i) {
    const int32_t id = (int32_t)(first + i);
    push_flow(fab, inst, src[i], dst[i], bytes[i], start ? start[i] : 0.0, conn_id ? conn_id[i] : id);
    if (dep_off)
      for (int64_t e = dep_off[i]; e < dep_off[i + 1]; ++e) push_dep(inst, (int32_t)dep_ids[e]);
  }
  inst.flow_count += n;
  return PHS_OK;
}

// Compute spans: flows of duration * 2^32 work units over the engine link of (gpu, lane); src = dst = gpu marks them.
phs_status append_spans(const Fabric &fab, Instance &inst, int64_t n, const int32_t *gpu, const int32_t *lane,
                        const double *duration, const double *start, const int64_t *dep_off, const int64_t *dep_ids,
                        std::string *why) {
  auto bad = [&](const char *m) {
    if (why) *why = m;
    return PHS_EINVAL;
  };
  if (n < 0 || (n > 0 && (!gpu || !duration))) return bad("null span arrays");
  if (fab.compute_lanes() <= 0) return bad("the topology has no compute lanes (phs_topology_desc.compute_lanes)");
  expand_pending(fab, inst);  // flow ids follow submission order
  const int64_t first = inst.n_flows();
  if (first + n > 0x7ffffff0LL) {
    if (why) *why = "too many flows in one instance";
    return PHS_ERANGE;
  }
  for (int64_t i = 0; i < n; ++i) {
    if (gpu[i] < 0 || gpu[i] >= fab.n_gpus()) return bad("gpu out of range");
    if (lane && (lane[i] < 0 || lane[i] >= fab.compute_lanes())) return bad("lane out of range");
    if (!(duration[i] > 0.0) || !(duration[i] < 0x1p20)) return bad("duration_s must be in (0, 2^20)");
    if (start && (!(start[i] >= 0.0) || !std::isfinite(start[i]))) return bad("start_time_s must be >= 0 and finite");
    if (dep_off) {
      if (dep_off[i + 1] < dep_off[i]) return bad("dep_off must be non-decreasing");
      if (dep_off[i + 1] > dep_off[i] && !dep_ids) return bad("dep_flow_ids is null");
      for (int64_t e = dep_off[i]; e < dep_off[i + 1]; ++e)
        if (dep_ids[e] < 0 || dep_ids[e] >= first + i) return bad("a span may only depend on earlier flows");
    }
  }
  for (int64_t i = 0; i < n; ++i) {
    push_flow(fab, inst, gpu[i], gpu[i], duration[i] * 0x1p32, start ? start[i] : 0.0, lane ? lane[i] : 0);
    if (dep_off)
      for (int64_t e = dep_off[i]; e < dep_off[i + 1]; ++e) push_dep(inst, (int32_t)dep_ids[e]);
  }
  inst.flow_count += n;
  return PHS_OK;
}

}  // namespace phs
