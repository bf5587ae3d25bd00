/*
 * orc_netsim.c -- CPU ORACLE (test infrastructure, not product code).  See orc_netsim.h for the
 * passages of PAPER.md this follows and the pins that hold it.  Build: oracle/build_oracle.py
 * (gcc -O2 -ffp-contract=off; x86-64 SSE2 doubles, no x87, no FMA contraction).
 *
 * Section tags S0..S6 refer to DESIGN.md "Readings" (= SURVEY.md sec 8(c)).
 */
#include "orc_netsim.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ---- S0: units.  bytes, seconds, byte/s.  Rates live on a 2^-20 byte/s grid (reading R-FX). ---- */
#define FRAC_BITS 20
static int64_t rate_to_q(double Bps) { return (int64_t)floor(Bps * 1048576.0); } /* x * 2^20, floor */
static double q_to_rate(int64_t q) { return (double)q * 0x1p-20; }               /* RN conversion, exact scale */

enum { WAITING = 0, PENDING = 1, ACTIVE = 2, DONE = 3 };

typedef struct {
  int32_t kind, n, first_flow, n_flows, steps;
  int32_t chunks; /* pipeline chunks of the chain / tree kinds (1 for the ring kinds and the all-to-all) */
  int32_t *ranks;
} coll_t;

typedef struct {
  int64_t ev;
  int32_t flow;
  double rate, t0, t1;
} trace_row;

struct orc_sim {
  orc_topology_desc d;
  uint64_t seed;
  int32_t G, n_links, n_net_links, ran;
  /* ORC_TOPO_GRAPH: out-links of every node (CSR, ascending link id), endpoints, hop distance to every GPU */
  int32_t n_nodes, *adj_off, *adj, *l_from, *l_to, *dist;
  double *cap, *lat; /* per directed link */
  /* flows */
  int64_t F, Fcap;
  int32_t *src, *dst, *conn;
  double *bytes, *start, *Lat;
  int64_t *path_off; /* [F+1] */
  int32_t *path;
  int64_t path_cap;
  int64_t *pred_off; /* [F+1] */
  int32_t *pred;
  int64_t pred_cap;
  /* collectives */
  coll_t *coll;
  int32_t n_coll, coll_cap;
  /* results */
  double *t_done;
  int32_t *bneck;
  orc_event *ev;
  int64_t n_ev, ev_cap;
  trace_row *tr;
  int64_t n_tr, tr_cap;
  /* throughput history: one record per rate change of a flow */
  int32_t *h_flow;
  double *h_t, *h_rate;
  double *h_rem;     /* remaining bytes at h_t, after the settle (what a rollback restores, PAPER.md L128 / L167) */
  int64_t *h_ev;     /* loop iteration (= index of the event it precedes) that wrote the record */
  int64_t *h_rq;     /* the rate in quanta of 2^-20 byte/s (h_rate is its binary64 image, inexact above 2^53 quanta) */
  int64_t n_h, h_cap;
  int64_t *done_ev;  /* per flow: index of the event in which it completed, -1 if it has not */
  int64_t F_res;     /* flows t_done / bneck / done_ev are allocated for */
  int64_t gc_events; /* events below this index cannot be rolled back into any more (orc_gc) */
  double work[7];
};

/* NEXT-1 (defined with the event loop): events with t < T; forget the events from index K on */
static int64_t events_before(const orc_sim *s, double T);
static int32_t rollback_events(orc_sim *s, int64_t K);

/* ------------------------------------------------------------------ S1: topology & link numbering */
static int32_t nvl_up(int32_t g) { return 2 * g; }
static int32_t nvl_dn(int32_t g) { return 2 * g + 1; }
static int32_t nic_up(const orc_sim *s, int32_t g) { return 2 * s->G + 2 * g; }
static int32_t nic_dn(const orc_sim *s, int32_t g) { return 2 * s->G + 2 * g + 1; }
static int32_t base1(const orc_sim *s) { return 4 * s->G; }
/* leaf-spine: pair u = (leaf*n_spines + spine)*P + p */
static int32_t ls_pair(const orc_sim *s, int32_t leaf, int32_t spine, int32_t p) {
  return (leaf * s->d.n_spines + spine) * s->d.uplinks_per_leaf_spine + p;
}
/* fat tree tier1<->tier2: pair u = (pod*(k/2) + edge)*(k/2) + agg */
static int32_t ft_pair1(const orc_sim *s, int32_t pod, int32_t edge, int32_t agg) {
  int32_t h = s->d.k / 2;
  return (pod * h + edge) * h + agg;
}
static int32_t ft_npairs1(const orc_sim *s) { return s->d.k * (s->d.k / 2) * (s->d.k / 2); }
static int32_t base2(const orc_sim *s) { return base1(s) + 2 * ft_npairs1(s); }
/* fat tree tier2<->tier3: pair u = (pod*(k/2) + agg)*U + j ; core = agg*U + j */
static int32_t ft_pair2(const orc_sim *s, int32_t pod, int32_t agg, int32_t j) {
  return (pod * (s->d.k / 2) + agg) * s->d.agg_uplinks + j;
}

int32_t orc_create_topology(const orc_topology_desc *d, uint64_t seed, orc_sim **out) {
  if (!d || !out) return ORC_EINVAL;
  if (d->n_hosts <= 0 || d->gpus_per_host <= 0) return ORC_EINVAL;
  if (!(d->nvlink_Bps > 0) || !(d->nic_Bps > 0) || !(d->hop_latency_s >= 0)) return ORC_EINVAL;
  int64_t G = (int64_t)d->n_hosts * d->gpus_per_host;
  int64_t L = 4 * G;
  if (d->kind == ORC_TOPO_LEAF_SPINE) {
    if (d->n_leaves <= 0 || d->n_spines <= 0 || d->uplinks_per_leaf_spine <= 0) return ORC_EINVAL;
    if (d->n_hosts % d->n_leaves != 0 || !(d->fabric_Bps > 0)) return ORC_EINVAL;
    L += 2 * (int64_t)d->n_leaves * d->n_spines * d->uplinks_per_leaf_spine;
  } else if (d->kind == ORC_TOPO_FAT_TREE) {
    int32_t k = d->k;
    if (k < 2 || k % 2 != 0 || d->agg_uplinks <= 0 || !(d->fabric_Bps > 0)) return ORC_EINVAL;
    if (d->gpus_per_host != k / 2 || d->n_hosts != k * (k / 2)) return ORC_EINVAL;
    L += 2 * (int64_t)k * (k / 2) * (k / 2) + 2 * (int64_t)k * (k / 2) * d->agg_uplinks;
  } else if (d->kind != ORC_TOPO_SINGLE)
    return ORC_EINVAL;
  if (d->compute_lanes < 0 || d->compute_lanes > 64) return ORC_EINVAL;
  int64_t L_net = L;
  L += G * d->compute_lanes; /* S7: compute engine links after all network links */
  if (L > 0x3fffffff) return ORC_ERANGE;
  orc_sim *s = (orc_sim *)calloc(1, sizeof(orc_sim));
  if (!s) return ORC_ENOMEM;
  s->d = *d;
  s->seed = seed;
  s->G = (int32_t)G;
  s->n_links = (int32_t)L;
  s->cap = (double *)malloc(sizeof(double) * L);
  s->lat = (double *)malloc(sizeof(double) * L);
  s->path_off = (int64_t *)calloc(1, sizeof(int64_t));
  s->pred_off = (int64_t *)calloc(1, sizeof(int64_t));
  if (!s->cap || !s->lat || !s->path_off || !s->pred_off) {
    orc_destroy(s);
    return ORC_ENOMEM;
  }
  s->n_net_links = (int32_t)L_net;
  for (int64_t l = 0; l < L; l++) {
    s->lat[l] = l < L_net ? d->hop_latency_s : 0.0;
    s->cap[l] = l < 2 * G ? d->nvlink_Bps : l < 4 * G ? d->nic_Bps : l < L_net ? d->fabric_Bps : 0x1p32;
  }
  *out = s;
  return ORC_OK;
}

int32_t orc_create_topology_graph(int32_t G, int32_t N, int32_t Ln, const int32_t *from, const int32_t *to,
                                  const double *cap, const double *lat, int32_t lanes, uint64_t seed, orc_sim **out) {
  if (!out || !from || !to || !cap || !lat || G < 2 || N < G || Ln < 1 || lanes < 0 || lanes > 64) return ORC_EINVAL;
  for (int32_t i = 0; i < Ln; i++) {
    if (from[i] < 0 || from[i] >= N || to[i] < 0 || to[i] >= N || from[i] == to[i]) return ORC_EINVAL;
    if (!(cap[i] > 0) || !(cap[i] < 0x1p42) || !(lat[i] >= 0) || !(lat[i] < INFINITY)) return ORC_EINVAL;
  }
  int64_t L = (int64_t)Ln + (int64_t)G * lanes;
  if (L > 0x3fffffff) return ORC_ERANGE;
  orc_sim *s = (orc_sim *)calloc(1, sizeof(orc_sim));
  if (!s) return ORC_ENOMEM;
  s->d.kind = ORC_TOPO_GRAPH;
  s->d.n_hosts = G; s->d.gpus_per_host = 1; s->d.compute_lanes = lanes;
  s->seed = seed;
  s->G = G; s->n_nodes = N; s->n_links = (int32_t)L; s->n_net_links = Ln;
  s->cap = (double *)malloc(sizeof(double) * L);
  s->lat = (double *)malloc(sizeof(double) * L);
  s->path_off = (int64_t *)calloc(1, sizeof(int64_t));
  s->pred_off = (int64_t *)calloc(1, sizeof(int64_t));
  s->adj_off = (int32_t *)calloc(N + 1, sizeof(int32_t));
  s->adj = (int32_t *)malloc(sizeof(int32_t) * Ln);
  s->l_from = (int32_t *)malloc(sizeof(int32_t) * Ln);
  s->l_to = (int32_t *)malloc(sizeof(int32_t) * Ln);
  s->dist = (int32_t *)malloc(sizeof(int32_t) * (size_t)G * N);
  int32_t *q = (int32_t *)malloc(sizeof(int32_t) * N), *rin_off = (int32_t *)calloc(N + 1, sizeof(int32_t)),
          *rin = (int32_t *)malloc(sizeof(int32_t) * Ln);
  if (!s->cap || !s->lat || !s->path_off || !s->pred_off || !s->adj_off || !s->adj || !s->l_from || !s->l_to || !s->dist ||
      !q || !rin_off || !rin) {
    free(q); free(rin_off); free(rin);
    orc_destroy(s);
    return ORC_ENOMEM;
  }
  for (int64_t l = 0; l < L; l++) { s->cap[l] = l < Ln ? cap[l] : 0x1p32; s->lat[l] = l < Ln ? lat[l] : 0.0; }
  memcpy(s->l_from, from, sizeof(int32_t) * Ln);
  memcpy(s->l_to, to, sizeof(int32_t) * Ln);
  /* out-links per node in ascending link id (counting sort keeps the order), in-links likewise for the BFS */
  for (int32_t i = 0; i < Ln; i++) { s->adj_off[from[i] + 1]++; rin_off[to[i] + 1]++; }
  for (int32_t v = 0; v < N; v++) { s->adj_off[v + 1] += s->adj_off[v]; rin_off[v + 1] += rin_off[v]; }
  {
    int32_t *c1 = (int32_t *)malloc(sizeof(int32_t) * N), *c2 = (int32_t *)malloc(sizeof(int32_t) * N);
    if (!c1 || !c2) { free(c1); free(c2); free(q); free(rin_off); free(rin); orc_destroy(s); return ORC_ENOMEM; }
    memcpy(c1, s->adj_off, sizeof(int32_t) * N);
    memcpy(c2, rin_off, sizeof(int32_t) * N);
    for (int32_t i = 0; i < Ln; i++) { s->adj[c1[from[i]]++] = i; rin[c2[to[i]]++] = i; }
    free(c1); free(c2);
  }
  /* dist[g][v] = links on a shortest path v -> GPU g (breadth-first search from g over the reversed links) */
  for (int32_t g = 0; g < G; g++) {
    int32_t *dg = s->dist + (size_t)g * N;
    for (int32_t v = 0; v < N; v++) dg[v] = -1;
    int32_t head = 0, tail = 0;
    dg[g] = 0; q[tail++] = g;
    while (head < tail) {
      int32_t v = q[head++];
      for (int32_t e = rin_off[v]; e < rin_off[v + 1]; e++) {
        int32_t u = from[rin[e]];
        if (dg[u] < 0) { dg[u] = dg[v] + 1; q[tail++] = u; }
      }
    }
  }
  free(q); free(rin_off); free(rin);
  *out = s;
  return ORC_OK;
}

void orc_destroy(orc_sim *s) {
  if (!s) return;
  for (int32_t c = 0; c < s->n_coll; c++) free(s->coll[c].ranks);
  free(s->adj_off); free(s->adj); free(s->l_from); free(s->l_to); free(s->dist);
  free(s->coll); free(s->cap); free(s->lat); free(s->src); free(s->dst); free(s->conn); free(s->bytes);
  free(s->start); free(s->Lat); free(s->path_off); free(s->path); free(s->pred_off); free(s->pred);
  free(s->t_done); free(s->bneck); free(s->ev); free(s->tr);
  free(s->h_flow); free(s->h_t); free(s->h_rate); free(s->h_rem); free(s->h_ev); free(s->h_rq); free(s->done_ev);
  free(s);
}

int32_t orc_num_links(const orc_sim *s, int32_t *out) {
  if (!s || !out) return ORC_EINVAL;
  *out = s->n_links;
  return ORC_OK;
}
int32_t orc_set_link_capacities(orc_sim *s, const double *c) {
  if (!s || !c) return ORC_EINVAL;
  if (s->ran) return ORC_ESTATE;
  for (int32_t l = 0; l < s->n_links; l++)
    if (!(c[l] > 0) || !(c[l] < 0x1p42)) return ORC_EINVAL;
  memcpy(s->cap, c, sizeof(double) * s->n_links);
  return ORC_OK;
}
int32_t orc_get_link_capacities(const orc_sim *s, double *c) {
  if (!s || !c) return ORC_EINVAL;
  memcpy(c, s->cap, sizeof(double) * s->n_links);
  return ORC_OK;
}

/* ------------------------------------------------------------------ S2: seeded ECMP routing */
uint64_t orc_mix64(uint64_t x) { /* SplitMix64 step (Steele, Lea, Flood 2014) */
  uint64_t z = x + 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

/* writes the path of (src,dst,conn) into p[0..5], returns its length */
static int32_t route(const orc_sim *s, int32_t src, int32_t dst, int32_t conn, int32_t *p) {
  const orc_topology_desc *d = &s->d;
  if (src == dst) { /* S7: a compute span; conn is its lane */
    p[0] = s->n_net_links + src * d->compute_lanes + conn;
    return 1;
  }
  if (d->kind == ORC_TOPO_GRAPH) { /* S8: hop by hop along shortest paths, seeded choice among the candidates */
    uint64_t Hg = orc_mix64(orc_mix64(orc_mix64(orc_mix64(s->seed) ^ (uint64_t)(uint32_t)src) ^ (uint64_t)(uint32_t)dst) ^
                            (uint64_t)(uint32_t)conn);
    const int32_t *dg = s->dist + (size_t)dst * s->n_nodes;
    int32_t u = src, k = 0;
    if (dg[u] < 0 || dg[u] > 6) return -1; /* unreachable / too long */
    while (u != dst) {
      int32_t cand[64], nc = 0;
      for (int32_t e = s->adj_off[u]; e < s->adj_off[u + 1]; e++)
        if (dg[s->l_to[s->adj[e]]] == dg[u] - 1 && nc < 64) cand[nc++] = s->adj[e];
      int32_t l = cand[orc_mix64(Hg ^ (uint64_t)(k + 1)) % (uint64_t)nc];
      p[k++] = l;
      u = s->l_to[l];
    }
    return k;
  }
  int32_t hs = src / d->gpus_per_host, hd = dst / d->gpus_per_host;
  if (hs == hd) {
    p[0] = nvl_up(src);
    p[1] = nvl_dn(dst);
    return 2;
  }
  uint64_t H = orc_mix64(orc_mix64(orc_mix64(orc_mix64(s->seed) ^ (uint64_t)(uint32_t)src) ^ (uint64_t)(uint32_t)dst) ^
                         (uint64_t)(uint32_t)conn);
  if (d->kind == ORC_TOPO_SINGLE) {
    p[0] = nic_up(s, src);
    p[1] = nic_dn(s, dst);
    return 2;
  }
  if (d->kind == ORC_TOPO_LEAF_SPINE) {
    int32_t per = d->n_hosts / d->n_leaves, ls = hs / per, ld = hd / per, P = d->uplinks_per_leaf_spine;
    if (ls == ld) {
      p[0] = nic_up(s, src);
      p[1] = nic_dn(s, dst);
      return 2;
    }
    int32_t c = (int32_t)(H % (uint64_t)(d->n_spines * P));
    int32_t spine = c / P, pu = c % P, pd = (int32_t)((H >> 32) % (uint64_t)P);
    p[0] = nic_up(s, src);
    p[1] = base1(s) + 2 * ls_pair(s, ls, spine, pu);     /* up: leaf_s -> spine */
    p[2] = base1(s) + 2 * ls_pair(s, ld, spine, pd) + 1; /* down: spine -> leaf_d */
    p[3] = nic_dn(s, dst);
    return 4;
  }
  /* fat tree: host == edge switch; pod = host / (k/2); edge = host % (k/2) */
  int32_t h = d->k / 2, qs = hs / h, es = hs % h, qd = hd / h, ed = hd % h;
  int32_t a = (int32_t)(H % (uint64_t)h);
  if (qs == qd) {
    p[0] = nic_up(s, src);
    p[1] = base1(s) + 2 * ft_pair1(s, qs, es, a);
    p[2] = base1(s) + 2 * ft_pair1(s, qd, ed, a) + 1;
    p[3] = nic_dn(s, dst);
    return 4;
  }
  int32_t j = (int32_t)((H >> 32) % (uint64_t)d->agg_uplinks);
  p[0] = nic_up(s, src);
  p[1] = base1(s) + 2 * ft_pair1(s, qs, es, a);
  p[2] = base2(s) + 2 * ft_pair2(s, qs, a, j);
  p[3] = base2(s) + 2 * ft_pair2(s, qd, a, j) + 1;
  p[4] = base1(s) + 2 * ft_pair1(s, qd, ed, a) + 1;
  p[5] = nic_dn(s, dst);
  return 6;
}

/* graph topologies: is there a route of at most 6 links?  (the presets always have one) */
static int routable(const orc_sim *s, int32_t src, int32_t dst) {
  if (s->d.kind != ORC_TOPO_GRAPH || src == dst) return 1;
  int32_t dd = s->dist[(size_t)dst * s->n_nodes + src];
  return dd >= 1 && dd <= 6;
}

/* ------------------------------------------------------------------ flow table growth */
static int grow_flows(orc_sim *s, int64_t need) {
  if (need <= s->Fcap) return 0;
  int64_t c = s->Fcap ? s->Fcap : 64;
  while (c < need) c *= 2;
#define RE(p, T, n)                               \
  do {                                            \
    void *q = realloc(p, sizeof(T) * (size_t)(n)); \
    if (!q) return -1;                            \
    p = (T *)q;                                   \
  } while (0)
  RE(s->src, int32_t, c); RE(s->dst, int32_t, c); RE(s->conn, int32_t, c);
  RE(s->bytes, double, c); RE(s->start, double, c); RE(s->Lat, double, c);
  RE(s->path_off, int64_t, c + 1); RE(s->pred_off, int64_t, c + 1);
  s->Fcap = c;
  return 0;
}
static int push_pred(orc_sim *s, int32_t p) {
  int64_t n = s->pred_off[s->F + 1];
  if (n + 1 > s->pred_cap) {
    int64_t c = s->pred_cap ? s->pred_cap * 2 : 256;
    RE(s->pred, int32_t, c);
    s->pred_cap = c;
  }
  s->pred[n] = p;
  s->pred_off[s->F + 1] = n + 1;
  return 0;
}
/* start a new flow record (id = s->F); preds are pushed with push_pred, then commit_flow */
static int begin_flow(orc_sim *s, int32_t src, int32_t dst, double bytes, double start, int32_t conn) {
  if (grow_flows(s, s->F + 1)) return -1;
  int64_t f = s->F;
  s->src[f] = src; s->dst[f] = dst; s->bytes[f] = bytes; s->start[f] = start; s->conn[f] = conn;
  int32_t p[6];
  int32_t h = route(s, src, dst, conn, p);
  if (h < 0) return -2; /* no route of at most 6 links (graph topologies) */
  int64_t po = s->path_off[f];
  if (po + h > s->path_cap) {
    int64_t c = s->path_cap ? s->path_cap * 2 : 256;
    RE(s->path, int32_t, c);
    s->path_cap = c;
  }
  double L = 0.0; /* S2: left-to-right sum of link latencies */
  for (int32_t i = 0; i < h; i++) {
    s->path[po + i] = p[i];
    L = L + s->lat[p[i]];
  }
  s->Lat[f] = L;
  s->path_off[f + 1] = po + h;
  s->pred_off[f + 1] = s->pred_off[f];
  return 0;
}
static void commit_flow(orc_sim *s) { s->F++; }

/* ------------------------------------------------------------------ S3: collective -> flows + DAG */
static int32_t coll_steps(int32_t kind, int32_t N) {
  return kind == ORC_ALLREDUCE_RING ? 2 * (N - 1) : kind == ORC_ALLTOALL ? 1 : N - 1;
}
/* id of the flow of collective c's last step that rank rho SENDS / RECEIVES in the ring; -1 if rho not in c */
static int32_t ring_index_of(const coll_t *c, int32_t rho) {
  for (int32_t i = 0; i < c->n; i++)
    if (c->ranks[i] == rho) return i;
  return -1;
}

/* S3, `after` edges.  F_A(rho) = the flows of collective A that must have finished before rank rho may start a
 * later collective: ring kinds: A's last-step flow sent by rho and the one received by rho; all-to-all: every flow
 * from / to rho; chain and tree kinds: the flows of A's LAST chunk that rho sends or receives.  rho not in A: none.
 * The flows of A are in the flow table already, so the chain / tree case simply looks at their endpoints. */
static int push_after_edges(orc_sim *s, const int32_t *after, int32_t n_after, int32_t rho) {
  for (int32_t a = 0; a < n_after; a++) {
    const coll_t *A = &s->coll[after[a]];
    int32_t ia = ring_index_of(A, rho);
    if (ia < 0) continue;
    if (A->kind == ORC_ALLTOALL) {
      for (int32_t x = 0; x < A->n; x++) {
        if (x == ia) continue;
        /* flow ia->x is entry (ia, x) of the row-major list without the diagonal */
        if (push_pred(s, A->first_flow + ia * (A->n - 1) + (x < ia ? x : x - 1))) return -1;
        if (push_pred(s, A->first_flow + x * (A->n - 1) + (ia < x ? ia : ia - 1))) return -1;
      }
    } else if (A->kind <= ORC_REDUCESCATTER_RING) {
      int32_t last = A->first_flow + (A->steps - 1) * A->n;
      if (push_pred(s, last + ia)) return -1;                    /* sent by rho */
      if (push_pred(s, last + (ia + A->n - 1) % A->n)) return -1; /* received by rho */
    } else {
      int32_t per_chunk = A->n_flows / A->chunks;
      for (int32_t f = A->first_flow + (A->chunks - 1) * per_chunk; f < A->first_flow + A->n_flows; f++)
        if (s->src[f] == rho || s->dst[f] == rho)
          if (push_pred(s, f)) return -1;
    }
  }
  return 0;
}

int32_t orc_add_collective(orc_sim *s, int32_t kind, const int32_t *ranks, int32_t N, double bytes, double start,
                           const int32_t *after, int32_t n_after, int32_t *out_id) {
  return orc_add_collective_ex(s, kind, ranks, N, bytes, start, after, n_after, 1, out_id);
}

/* S3 with the NEXT-3 kinds ("the communication patterns of different collective operations").
 * `chunks` = C >= 1 pipeline chunks of the chain / tree kinds (must be 1 for the ring kinds and the all-to-all):
 *   ORC_BROADCAST_CHAIN   root r[0]; hop i = 0..N-2 is r[i] -> r[i+1]; flow (c, i), id first + c (N-1) + i, carries
 *                         bytes / C; it waits for (c, i-1) (the chunk has arrived at r[i]) and (c-1, i) (sender FIFO).
 *   ORC_REDUCE_CHAIN      the same towards the root: hop i is r[N-1-i] -> r[N-2-i].
 *   ORC_ALLREDUCE_TREE    binary tree in heap order over the positions (parent(i) = (i-1)/2); per chunk c a block of
 *                         2 (N-1) flows: up(c, i), i = 1..N-1, id first + c 2(N-1) + (i-1), r[i] -> r[parent(i)],
 *                         waits for up(c, 2i+1), up(c, 2i+2) (the subtree's partial sums) and up(c-1, i) (FIFO);
 *                         down(c, i), id first + c 2(N-1) + (N-1) + (i-1), r[parent(i)] -> r[i], waits for
 *                         down(c, parent(i)) -- or, below the root, for up(c, 1) and up(c, 2) -- and down(c-1, i).
 * `start` and the `after` edges apply to every flow that has no predecessor inside the collective. */
int32_t orc_add_collective_ex(orc_sim *s, int32_t kind, const int32_t *ranks, int32_t N, double bytes, double start,
                              const int32_t *after, int32_t n_after, int32_t chunks, int32_t *out_id) {
  return orc_add_collective_full(s, kind, ranks, N, bytes, start, after, n_after, NULL, 0, chunks, out_id);
}

int32_t orc_add_collective_full(orc_sim *s, int32_t kind, const int32_t *ranks, int32_t N, double bytes, double start,
                                const int32_t *after, int32_t n_after, const int64_t *after_flows, int32_t n_after_flows,
                                int32_t chunks, int32_t *out_id) {
  if (!s || !ranks) return ORC_EINVAL;
  /* submitted after the simulation has run past its start time (L124): roll back to that time first */
  if (s->n_ev > 0 && start >= 0 && rollback_events(s, events_before(s, start)) != ORC_OK) return ORC_EINVAL;
  if (n_after_flows < 0 || (n_after_flows > 0 && !after_flows)) return ORC_EINVAL;
  for (int32_t k = 0; k < n_after_flows; k++)
    if (after_flows[k] < 0 || after_flows[k] >= s->F) return ORC_EINVAL; /* only flows submitted before */
  if (kind < 0 || kind > ORC_ALLREDUCE_TREE || N < 2 || !(bytes > 0) || !(bytes < INFINITY) || !(start >= 0) ||
      !(start < INFINITY))
    return ORC_EINVAL;
  if (chunks < 1 || chunks > 65536 || (kind <= ORC_ALLTOALL && chunks != 1)) return ORC_EINVAL;
  if (n_after < 0 || (n_after > 0 && !after)) return ORC_EINVAL;
  for (int32_t i = 0; i < N; i++) {
    if (ranks[i] < 0 || ranks[i] >= s->G) return ORC_EINVAL;
    for (int32_t j = 0; j < i; j++)
      if (ranks[j] == ranks[i]) return ORC_EINVAL;
  }
  for (int32_t a = 0; a < n_after; a++)
    if (after[a] < 0 || after[a] >= s->n_coll) return ORC_EINVAL;
  if (s->d.kind == ORC_TOPO_GRAPH) /* every pair of its ranks must be routable, whatever pairs the kind uses */
    for (int32_t i = 0; i < N; i++)
      for (int32_t j = 0; j < N; j++)
        if (!routable(s, ranks[i], ranks[j])) return ORC_EINVAL;
  int32_t S = coll_steps(kind, N);
  int64_t nf = kind == ORC_ALLTOALL ? (int64_t)N * (N - 1)
             : kind == ORC_ALLREDUCE_TREE ? (int64_t)chunks * 2 * (N - 1)
             : kind >= ORC_BROADCAST_CHAIN ? (int64_t)chunks * (N - 1)
                                           : (int64_t)S * N;
  if (s->F + nf > 0x7ffffff0) return ORC_ERANGE;
  if (s->n_coll == s->coll_cap) {
    int32_t c = s->coll_cap ? 2 * s->coll_cap : 16;
    void *q = realloc(s->coll, sizeof(coll_t) * c);
    if (!q) return ORC_ENOMEM;
    s->coll = (coll_t *)q;
    s->coll_cap = c;
  }
  int32_t cid = s->n_coll;
  coll_t *c = &s->coll[cid];
  c->kind = kind; c->n = N; c->first_flow = (int32_t)s->F; c->n_flows = (int32_t)nf; c->steps = S; c->chunks = chunks;
  c->ranks = (int32_t *)malloc(sizeof(int32_t) * N);
  if (!c->ranks) return ORC_ENOMEM;
  memcpy(c->ranks, ranks, sizeof(int32_t) * N);
  s->n_coll++; /* (ranks now owned by the table) */
  int32_t first = c->first_flow;
  /* edges of an initial flow sent by rho: the `after` collectives, then the listed flows / spans that touch rho */
#define PUSH_AFTER(rho)                                                              \
  do {                                                                               \
    if (push_after_edges(s, after, n_after, (rho))) return ORC_ENOMEM;               \
    for (int32_t k_ = 0; k_ < n_after_flows; k_++)                                   \
      if (s->src[after_flows[k_]] == (rho) || s->dst[after_flows[k_]] == (rho))      \
        if (push_pred(s, (int32_t)after_flows[k_])) return ORC_ENOMEM;               \
  } while (0)

  if (kind == ORC_ALLTOALL) {
    double chunk = bytes / (double)N; /* S3: one f64 division */
    for (int32_t i = 0; i < N; i++)
      for (int32_t j = 0; j < N; j++) {
        if (i == j) continue;
        if (begin_flow(s, ranks[i], ranks[j], chunk, start, cid)) return ORC_ENOMEM;
        PUSH_AFTER(ranks[i]);
        commit_flow(s);
      }
  } else if (kind <= ORC_REDUCESCATTER_RING) {
    double chunk = bytes / (double)N; /* S3: one f64 division */
    for (int32_t st = 0; st < S; st++)
      for (int32_t i = 0; i < N; i++) { /* flow (st,i): r[i] -> r[(i+1) mod N] */
        if (begin_flow(s, ranks[i], ranks[(i + 1) % N], chunk, st == 0 ? start : 0.0, cid)) return ORC_ENOMEM;
        if (st == 0) {
          PUSH_AFTER(ranks[i]);
        } else {
          if (push_pred(s, first + (st - 1) * N + (i + N - 1) % N)) return ORC_ENOMEM; /* data has arrived */
          if (push_pred(s, first + (st - 1) * N + i)) return ORC_ENOMEM;               /* sender FIFO */
        }
        commit_flow(s);
      }
  } else if (kind == ORC_BROADCAST_CHAIN || kind == ORC_REDUCE_CHAIN) {
    double piece = bytes / (double)chunks;
    for (int32_t ch = 0; ch < chunks; ch++)
      for (int32_t i = 0; i < N - 1; i++) {
        int32_t from = kind == ORC_BROADCAST_CHAIN ? ranks[i] : ranks[N - 1 - i];
        int32_t to = kind == ORC_BROADCAST_CHAIN ? ranks[i + 1] : ranks[N - 2 - i];
        int no_pred = ch == 0 && i == 0;
        if (begin_flow(s, from, to, piece, no_pred ? start : 0.0, cid)) return ORC_ENOMEM;
        if (no_pred) PUSH_AFTER(from);
        if (i > 0 && push_pred(s, first + ch * (N - 1) + i - 1)) return ORC_ENOMEM;  /* the chunk has arrived */
        if (ch > 0 && push_pred(s, first + (ch - 1) * (N - 1) + i)) return ORC_ENOMEM; /* sender FIFO */
        commit_flow(s);
      }
  } else { /* ORC_ALLREDUCE_TREE */
    double piece = bytes / (double)chunks;
    int32_t per = 2 * (N - 1);
    for (int32_t ch = 0; ch < chunks; ch++) {
      for (int32_t i = 1; i < N; i++) { /* up(ch, i): r[i] -> r[parent(i)] */
        int32_t l = 2 * i + 1, r = 2 * i + 2;
        int no_pred = ch == 0 && l >= N; /* a leaf's first chunk */
        if (begin_flow(s, ranks[i], ranks[(i - 1) / 2], piece, no_pred ? start : 0.0, cid)) return ORC_ENOMEM;
        if (no_pred) PUSH_AFTER(ranks[i]);
        if (l < N && push_pred(s, first + ch * per + (l - 1))) return ORC_ENOMEM;
        if (r < N && push_pred(s, first + ch * per + (r - 1))) return ORC_ENOMEM;
        if (ch > 0 && push_pred(s, first + (ch - 1) * per + (i - 1))) return ORC_ENOMEM;
        commit_flow(s);
      }
      for (int32_t i = 1; i < N; i++) { /* down(ch, i): r[parent(i)] -> r[i] */
        int32_t p = (i - 1) / 2;
        if (begin_flow(s, ranks[p], ranks[i], piece, 0.0, cid)) return ORC_ENOMEM;
        if (p == 0) { /* the root holds the full sum of the chunk once its children's partial sums are in */
          if (push_pred(s, first + ch * per + 0)) return ORC_ENOMEM;
          if (N > 2 && push_pred(s, first + ch * per + 1)) return ORC_ENOMEM;
        } else if (push_pred(s, first + ch * per + (N - 1) + (p - 1))) return ORC_ENOMEM;
        if (ch > 0 && push_pred(s, first + (ch - 1) * per + (N - 1) + (i - 1))) return ORC_ENOMEM;
        commit_flow(s);
      }
    }
  }
#undef PUSH_AFTER
  if (out_id) *out_id = cid;
  return ORC_OK;
}

int32_t orc_add_flows(orc_sim *s, int64_t n, const int32_t *src, const int32_t *dst, const double *bytes,
                      const double *start, const int64_t *dep_off, const int64_t *dep_ids, const int32_t *conn_id,
                      int64_t *out_first) {
  if (!s || n < 0 || (n > 0 && (!src || !dst || !bytes))) return ORC_EINVAL;
  if (s->F + n > 0x7ffffff0) return ORC_ERANGE;
  int64_t first = s->F;
  if (s->n_ev > 0 && n > 0) { /* late submission (L124): roll back to the earliest new start time */
    double T2 = INFINITY;
    for (int64_t i = 0; i < n; i++) { double st = start ? start[i] : 0.0; if (st < T2) T2 = st; }
    if (!(T2 >= 0) || rollback_events(s, events_before(s, T2)) != ORC_OK) return ORC_EINVAL;
  }
  for (int64_t i = 0; i < n; i++) { /* validate everything before mutating */
    if (src[i] < 0 || src[i] >= s->G || dst[i] < 0 || dst[i] >= s->G || src[i] == dst[i]) return ORC_EINVAL;
    if (!routable(s, src[i], dst[i])) return ORC_EINVAL;
    if (!(bytes[i] > 0) || !(bytes[i] < INFINITY)) return ORC_EINVAL;
    if (start && (!(start[i] >= 0) || !(start[i] < INFINITY))) return ORC_EINVAL;
    if (dep_off) {
      if (dep_off[i + 1] < dep_off[i] || (dep_off[i + 1] > dep_off[i] && !dep_ids)) return ORC_EINVAL;
      for (int64_t e = dep_off[i]; e < dep_off[i + 1]; e++)
        if (dep_ids[e] < 0 || dep_ids[e] >= first + i) return ORC_EINVAL; /* only earlier flows */
    }
  }
  for (int64_t i = 0; i < n; i++) {
    int32_t conn = conn_id ? conn_id[i] : (int32_t)(first + i);
    if (begin_flow(s, src[i], dst[i], bytes[i], start ? start[i] : 0.0, conn)) return ORC_ENOMEM;
    if (dep_off)
      for (int64_t e = dep_off[i]; e < dep_off[i + 1]; e++)
        if (push_pred(s, (int32_t)dep_ids[e])) return ORC_ENOMEM;
    commit_flow(s);
  }
  if (out_first) *out_first = first;
  return ORC_OK;
}

/* S7: compute spans = flows of duration * 2^32 work units over the engine link of (gpu, lane) */
int32_t orc_add_spans(orc_sim *s, int64_t n, const int32_t *gpu, const int32_t *lane, const double *duration,
                      const double *start, const int64_t *dep_off, const int64_t *dep_ids, int64_t *out_first) {
  if (!s || n < 0 || (n > 0 && (!gpu || !duration))) return ORC_EINVAL;
  if (s->d.compute_lanes <= 0) return ORC_EINVAL;
  if (s->F + n > 0x7ffffff0) return ORC_ERANGE;
  int64_t first = s->F;
  if (s->n_ev > 0 && n > 0) { /* late submission (L124): roll back to the earliest new start time */
    double T2 = INFINITY;
    for (int64_t i = 0; i < n; i++) { double st = start ? start[i] : 0.0; if (st < T2) T2 = st; }
    if (!(T2 >= 0) || rollback_events(s, events_before(s, T2)) != ORC_OK) return ORC_EINVAL;
  }
  for (int64_t i = 0; i < n; i++) {
    if (gpu[i] < 0 || gpu[i] >= s->G) return ORC_EINVAL;
    if (lane && (lane[i] < 0 || lane[i] >= s->d.compute_lanes)) return ORC_EINVAL;
    if (!(duration[i] > 0) || !(duration[i] < 0x1p20)) return ORC_EINVAL;
    if (start && (!(start[i] >= 0) || !(start[i] < INFINITY))) return ORC_EINVAL;
    if (dep_off) {
      if (dep_off[i + 1] < dep_off[i] || (dep_off[i + 1] > dep_off[i] && !dep_ids)) return ORC_EINVAL;
      for (int64_t e = dep_off[i]; e < dep_off[i + 1]; e++)
        if (dep_ids[e] < 0 || dep_ids[e] >= first + i) return ORC_EINVAL;
    }
  }
  for (int64_t i = 0; i < n; i++) {
    if (begin_flow(s, gpu[i], gpu[i], duration[i] * 0x1p32, start ? start[i] : 0.0, lane ? lane[i] : 0)) return ORC_ENOMEM;
    if (dep_off)
      for (int64_t e = dep_off[i]; e < dep_off[i + 1]; e++)
        if (push_pred(s, (int32_t)dep_ids[e])) return ORC_ENOMEM;
    commit_flow(s);
  }
  if (out_first) *out_first = first;
  return ORC_OK;
}

/* ------------------------------------------------------------------ S5: max-min progressive filling */
typedef struct {
  int32_t n_links;
  int64_t *cap_rem; /* remaining capacity, rate quanta */
  int32_t *n;       /* unfrozen active flows on the link */
  int32_t *k;       /* newly frozen flows crossing the link in this iteration */
  int32_t *touched;
  int64_t *adj_off; /* link -> active flows (indices into act[]) */
  int32_t *adj;
  int64_t adj_cap;
  uint8_t *frozen;
  int64_t frozen_cap;
  /* fast mode heap of (share, link) */
  int64_t *hs;
  int32_t *hl;
  int64_t hn, hcap;
} ws_t;

static void ws_free(ws_t *w) {
  free(w->cap_rem); free(w->n); free(w->k); free(w->touched); free(w->adj_off); free(w->adj); free(w->frozen);
  free(w->hs); free(w->hl);
}
static int ws_init(ws_t *w, int32_t L) {
  memset(w, 0, sizeof(*w));
  w->n_links = L;
  w->cap_rem = (int64_t *)malloc(sizeof(int64_t) * L);
  w->n = (int32_t *)calloc(L, sizeof(int32_t));
  w->k = (int32_t *)calloc(L, sizeof(int32_t));
  w->touched = (int32_t *)malloc(sizeof(int32_t) * L);
  w->adj_off = (int64_t *)malloc(sizeof(int64_t) * (L + 1));
  return (w->cap_rem && w->n && w->k && w->touched && w->adj_off) ? 0 : -1;
}
static int heap_less(const ws_t *w, int64_t a, int64_t b) {
  return w->hs[a] < w->hs[b] || (w->hs[a] == w->hs[b] && w->hl[a] < w->hl[b]);
}
static int heap_push(ws_t *w, int64_t s, int32_t l) {
  if (w->hn == w->hcap) {
    int64_t c = w->hcap ? 2 * w->hcap : 1024;
    void *a = realloc(w->hs, sizeof(int64_t) * c), *b;
    if (!a) return -1;
    w->hs = (int64_t *)a;
    b = realloc(w->hl, sizeof(int32_t) * c);
    if (!b) return -1;
    w->hl = (int32_t *)b;
    w->hcap = c;
  }
  int64_t i = w->hn++;
  w->hs[i] = s; w->hl[i] = l;
  while (i > 0) {
    int64_t p = (i - 1) / 2;
    if (!heap_less(w, i, p)) break;
    int64_t ts = w->hs[i]; w->hs[i] = w->hs[p]; w->hs[p] = ts;
    int32_t tl = w->hl[i]; w->hl[i] = w->hl[p]; w->hl[p] = tl;
    i = p;
  }
  return 0;
}
static void heap_pop(ws_t *w) {
  int64_t n = --w->hn, i = 0;
  w->hs[0] = w->hs[n]; w->hl[0] = w->hl[n];
  for (;;) {
    int64_t a = 2 * i + 1, b = a + 1, m = i;
    if (a < n && heap_less(w, a, m)) m = a;
    if (b < n && heap_less(w, b, m)) m = b;
    if (m == i) break;
    int64_t ts = w->hs[i]; w->hs[i] = w->hs[m]; w->hs[m] = ts;
    int32_t tl = w->hl[i]; w->hl[i] = w->hl[m]; w->hl[m] = tl;
    i = m;
  }
}

/* Active flows act[0..nA) (ids into the path CSR).  Outputs indexed by flow id.  Returns the number of
 * links with n>0 at the start (Lambda_act) through *lam_act. */
static int solve_maxmin(ws_t *w, const int64_t *capq, int32_t nA, const int32_t *act, const int64_t *path_off,
                        const int32_t *path, int32_t mode, int64_t *rq, int32_t *bneck, int32_t *n_rounds,
                        int32_t *first_bneck, int32_t *lam_act) {
  int32_t L = w->n_links;
  *n_rounds = 0; *first_bneck = -1; *lam_act = 0;
  if (nA == 0) return 0;
  /* init: cap_rem = cap, n = # active flows on the link, all unfrozen (S5) */
  for (int32_t l = 0; l < L; l++) { w->cap_rem[l] = capq[l]; w->n[l] = 0; }
  int64_t tot = 0;
  for (int32_t a = 0; a < nA; a++)
    for (int64_t e = path_off[act[a]]; e < path_off[act[a] + 1]; e++) { w->n[path[e]]++; tot++; }
  if (tot > w->adj_cap) {
    void *q = realloc(w->adj, sizeof(int32_t) * tot);
    if (!q) return -1;
    w->adj = (int32_t *)q; w->adj_cap = tot;
  }
  if (nA > w->frozen_cap) {
    void *q = realloc(w->frozen, nA);
    if (!q) return -1;
    w->frozen = (uint8_t *)q; w->frozen_cap = nA;
  }
  memset(w->frozen, 0, nA);
  w->adj_off[0] = 0;
  for (int32_t l = 0; l < L; l++) { w->adj_off[l + 1] = w->adj_off[l] + w->n[l]; if (w->n[l] > 0) (*lam_act)++; }
  { /* fill link -> active-flow lists */
    int64_t *cur = (int64_t *)malloc(sizeof(int64_t) * L);
    if (!cur) return -1;
    memcpy(cur, w->adj_off, sizeof(int64_t) * L);
    for (int32_t a = 0; a < nA; a++)
      for (int64_t e = path_off[act[a]]; e < path_off[act[a] + 1]; e++) w->adj[cur[path[e]]++] = a;
    free(cur);
  }
  if (mode == ORC_MODE_FAST) {
    w->hn = 0;
    for (int32_t l = 0; l < L; l++)
      if (w->n[l] > 0 && heap_push(w, w->cap_rem[l] / w->n[l], l)) return -1;
  }
  int32_t unfrozen = nA;
  while (unfrozen > 0) {
    /* the bottleneck link: smallest share = cap_rem / n over links with n > 0; ties -> lowest link id */
    int32_t b = -1;
    int64_t s = 0;
    if (mode == ORC_MODE_NAIVE) {
      for (int32_t l = 0; l < L; l++) {
        if (w->n[l] <= 0) continue;
        int64_t sh = w->cap_rem[l] / w->n[l];
        if (b < 0 || sh < s) { b = l; s = sh; }
      }
    } else {
      for (;;) { /* lazy deletion: an entry is live iff it still equals the link's current share */
        int64_t sh = w->hs[0];
        int32_t l = w->hl[0];
        heap_pop(w);
        if (w->n[l] > 0 && w->cap_rem[l] / w->n[l] == sh) { b = l; s = sh; break; }
      }
    }
    if (*n_rounds == 0) *first_bneck = b;
    /* freeze every unfrozen active flow on b at rate s; count k[l] on all their links */
    int32_t nt = 0;
    for (int64_t e = w->adj_off[b]; e < w->adj_off[b + 1]; e++) {
      int32_t a = w->adj[e];
      if (w->frozen[a]) continue;
      w->frozen[a] = 1;
      rq[act[a]] = s;
      bneck[act[a]] = b;
      unfrozen--;
      for (int64_t pe = path_off[act[a]]; pe < path_off[act[a] + 1]; pe++) {
        int32_t l = path[pe];
        if (w->k[l]++ == 0) w->touched[nt++] = l;
      }
    }
    /* debit: cap_rem -= k*s ; n -= k */
    for (int32_t t = 0; t < nt; t++) {
      int32_t l = w->touched[t];
      w->cap_rem[l] = w->cap_rem[l] - (int64_t)w->k[l] * s;
      w->n[l] -= w->k[l];
      w->k[l] = 0;
      if (mode == ORC_MODE_FAST && w->n[l] > 0 && heap_push(w, w->cap_rem[l] / w->n[l], l)) return -1;
    }
    (*n_rounds)++;
  }
  return 0;
}

/* SURVEY.md 8(c) S5 exactly as written there (binary64 shares), one bottleneck link per iteration, dense argmin.
 * Kept beside the R-FX solver to measure how far the two readings are apart (tests: < 1e-9 relative on times). */
static int solve_maxmin_f64(ws_t *w, const double *cap, int32_t nA, const int32_t *act, const int64_t *path_off,
                            const int32_t *path, double *rate, int32_t *bneck, int32_t *n_rounds, int32_t *first_bneck,
                            int32_t *lam_act) {
  int32_t L = w->n_links;
  *n_rounds = 0; *first_bneck = -1; *lam_act = 0;
  if (nA == 0) return 0;
  double *cap_rem = (double *)malloc(sizeof(double) * L);
  if (!cap_rem) return -1;
  for (int32_t l = 0; l < L; l++) { cap_rem[l] = cap[l]; w->n[l] = 0; }
  if (nA > w->frozen_cap) {
    void *q = realloc(w->frozen, nA);
    if (!q) { free(cap_rem); return -1; }
    w->frozen = (uint8_t *)q; w->frozen_cap = nA;
  }
  memset(w->frozen, 0, nA);
  for (int32_t a = 0; a < nA; a++)
    for (int64_t e = path_off[act[a]]; e < path_off[act[a] + 1]; e++) w->n[path[e]]++;
  for (int32_t l = 0; l < L; l++) if (w->n[l] > 0) (*lam_act)++;
  int32_t unfrozen = nA;
  while (unfrozen > 0) {
    int32_t b = -1;
    double s = 0.0;
    for (int32_t l = 0; l < L; l++) {
      if (w->n[l] <= 0) continue;
      double sh = cap_rem[l] / (double)w->n[l];
      if (b < 0 || sh < s) { b = l; s = sh; }
    }
    if (*n_rounds == 0) *first_bneck = b;
    int32_t nt = 0;
    for (int32_t a = 0; a < nA; a++) { /* every unfrozen active flow crossing b */
      if (w->frozen[a]) continue;
      int on_b = 0;
      for (int64_t pe = path_off[act[a]]; pe < path_off[act[a] + 1]; pe++) if (path[pe] == b) on_b = 1;
      if (!on_b) continue;
      w->frozen[a] = 1;
      rate[act[a]] = s;
      bneck[act[a]] = b;
      unfrozen--;
      for (int64_t pe = path_off[act[a]]; pe < path_off[act[a] + 1]; pe++) {
        int32_t l = path[pe];
        if (w->k[l]++ == 0) w->touched[nt++] = l;
      }
    }
    for (int32_t t = 0; t < nt; t++) {
      int32_t l = w->touched[t];
      cap_rem[l] = cap_rem[l] - (double)w->k[l] * s;
      w->n[l] -= w->k[l];
      w->k[l] = 0;
    }
    (*n_rounds)++;
  }
  free(cap_rem);
  return 0;
}

int32_t orc_maxmin(int32_t n_links, const double *cap, int32_t n_flows, const int64_t *path_off, const int32_t *path,
                   int32_t mode, double *rate, int32_t *bneck, int32_t *n_rounds, int32_t *first_bneck) {
  if (n_links <= 0 || n_flows < 0 || !cap || !path_off || !rate || !bneck) return ORC_EINVAL;
  ws_t w;
  if (ws_init(&w, n_links)) { ws_free(&w); return ORC_ENOMEM; }
  int64_t *capq = (int64_t *)malloc(sizeof(int64_t) * n_links);
  int64_t *rq = (int64_t *)malloc(sizeof(int64_t) * (n_flows + 1));
  int32_t *act = (int32_t *)malloc(sizeof(int32_t) * (n_flows + 1));
  int32_t rc = ORC_OK, R = 0, fb = -1, lam = 0;
  if (!capq || !rq || !act) rc = ORC_ENOMEM;
  if (rc == ORC_OK) {
    for (int32_t l = 0; l < n_links; l++) capq[l] = rate_to_q(cap[l]);
    for (int32_t f = 0; f < n_flows; f++) act[f] = f;
    if (solve_maxmin(&w, capq, n_flows, act, path_off, path, mode, rq, bneck, &R, &fb, &lam)) rc = ORC_ENOMEM;
  }
  if (rc == ORC_OK) {
    for (int32_t f = 0; f < n_flows; f++) rate[f] = q_to_rate(rq[f]);
    if (n_rounds) *n_rounds = R;
    if (first_bneck) *first_bneck = fb;
  }
  free(capq); free(rq); free(act); ws_free(&w);
  return rc;
}

/* ------------------------------------------------------------------ NEXT-1: time rollback
 * The simulator may have run ahead (to T1) when something arrives with an earlier timestamp T2.  Rolling back keeps
 * the events before T2 and forgets the rest: completion times, bottlenecks and history records written from the first
 * dropped event on are discarded; the next run call rebuilds the state after the last kept event from the
 * throughput history (see orc_run_ex) and simulates forward again. */
static int64_t events_before(const orc_sim *s, double T) { /* events are in time order */
  int64_t k = 0;
  while (k < s->n_ev && s->ev[k].t < T) k++;
  return k;
}
static int32_t rollback_events(orc_sim *s, int64_t K) {
  if (K >= s->n_ev) return ORC_OK; /* nothing at or after that point has been simulated */
  if (K < s->gc_events) return ORC_EINVAL; /* the history below the watermark is gone */
  s->n_ev = K;
  for (int64_t f = 0; f < s->F_res; f++)
    if (s->done_ev[f] >= K) { s->done_ev[f] = -1; s->t_done[f] = NAN; s->bneck[f] = -1; }
  int64_t keep = 0;
  for (int64_t i = 0; i < s->n_h; i++)
    if (s->h_ev[i] < K) {
      s->h_flow[keep] = s->h_flow[i]; s->h_t[keep] = s->h_t[i]; s->h_rate[keep] = s->h_rate[i];
      s->h_rem[keep] = s->h_rem[i]; s->h_ev[keep] = s->h_ev[i]; s->h_rq[keep] = s->h_rq[i];
      keep++;
    }
  s->n_h = keep;
  return ORC_OK;
}
/* everything from time T on is forgotten (events with t < T stay) */
int32_t orc_rollback(orc_sim *s, double T) {
  if (!s || !(T >= 0)) return ORC_EINVAL;
  return rollback_events(s, events_before(s, T));
}
/* "updating the start time of an existing flow" (L167): rolls back to min(old, new) start time, then changes it */
int32_t orc_update_flow_start(orc_sim *s, int64_t flow, double start) {
  if (!s || flow < 0 || flow >= s->F || !(start >= 0) || !(start < INFINITY)) return ORC_EINVAL;
  /* The start time acts through t_act = max(start, release) + Lat, release = completion of the flow's last
   * predecessor (0 without predecessors).  If the flow has not been released in what was simulated so far, its start
   * time has not been used yet; otherwise the past differs from max(old, release) or max(new, release) on, whichever is
   * earlier -- unless the two are equal. */
  double rel = 0.0;
  int released = 1;
  for (int64_t e = s->pred_off[flow]; e < s->pred_off[flow + 1]; e++) {
    int32_t p = s->pred[e];
    if (p >= s->F_res || s->done_ev[p] < 0) { released = 0; break; }
    if (s->t_done[p] > rel) rel = s->t_done[p];
  }
  if (released && s->n_ev > 0) {
    double a = s->start[flow] > rel ? s->start[flow] : rel, b = start > rel ? start : rel;
    if (a != b) {
      int32_t rc = rollback_events(s, events_before(s, a < b ? a : b));
      if (rc != ORC_OK) return rc;
    }
  }
  s->start[flow] = start;
  return ORC_OK;
}
/* garbage collection (L130): nothing will ever be rolled back to a time before T, so every flow keeps only the last
 * of its history records older than that; later rollbacks to times >= T are unaffected */
int32_t orc_gc(orc_sim *s, double T) {
  if (!s || !(T >= 0)) return ORC_EINVAL;
  int64_t K = events_before(s, T);
  if (K <= s->gc_events) return ORC_OK;
  int64_t *last = (int64_t *)malloc(sizeof(int64_t) * (s->F + 1));
  if (!last) return ORC_ENOMEM;
  for (int64_t f = 0; f < s->F; f++) last[f] = -1;
  for (int64_t i = 0; i < s->n_h; i++)
    if (s->h_ev[i] < K) last[s->h_flow[i]] = i;
  int64_t keep = 0;
  for (int64_t i = 0; i < s->n_h; i++) {
    int32_t f = s->h_flow[i];
    if (s->h_ev[i] < K && (last[f] != i || (s->done_ev[f] >= 0 && s->done_ev[f] < K))) continue; /* superseded / done */
    s->h_flow[keep] = s->h_flow[i]; s->h_t[keep] = s->h_t[i]; s->h_rate[keep] = s->h_rate[i];
    s->h_rem[keep] = s->h_rem[i]; s->h_ev[keep] = s->h_ev[i]; s->h_rq[keep] = s->h_rq[i];
    keep++;
  }
  s->n_h = keep;
  s->gc_events = K;
  free(last);
  return ORC_OK;
}

/* ------------------------------------------------------------------ S4: flow states & event loop */
/* S4.4 / Q11: remaining bytes after draining at `rate` for dt seconds: mul, then sub, then clamp at 0.  (Under
 * R-LZ the clamp is a guard: DESIGN.md sec 2 argues that a flow still active at `now` < tc cannot have drained
 * more than it holds; the function is exported so that the branch is pinned directly.) */
static double settle(double rem, double rate, double dt) {
  double m = rate * dt;
  double r = rem - m;
  return r > 0.0 ? r : 0.0;
}
double orc_settle(double rem, double rate_Bps, double dt) { return settle(rem, rate_Bps, dt); }

int32_t orc_run(orc_sim *s, int32_t mode, int32_t trace) { return orc_run_ex(s, mode, trace, INFINITY, 0); }
int32_t orc_run_until(orc_sim *s, int32_t mode, int32_t trace, double t_stop) {
  return orc_run_ex(s, mode, trace, t_stop, 0);
}

/* "advancing the simulation ... up to a specified time": the event loop stops before the first
 * event later than t_stop.  Flows that have not completed by then keep t_done = NaN and bneck = -1; the event
 * log and the throughput history hold what happened up to t_stop. */
/* flags (the two readings DESIGN.md sec 2 CHANGED, kept so that the change can be measured against the tolerance
 * BASELINE.json states, 1e-9 relative): ORC_FLAG_SETTLE_EVERY_EVENT = SURVEY.md 8(c) S4.4 as written (every ACTIVE
 * flow is debited at every event: rem = max(rem - rate*dt, 0), tc = now + rem/rate) instead of R-LZ;
 * ORC_FLAG_F64_SHARES = SURVEY.md 8(c) S5 as written (cap_rem and share are binary64: share = cap_rem / n,
 * cap_rem -= k * share) instead of R-FX.  Neither is used by any parity test of the CUDA path. */
int32_t orc_run_ex(orc_sim *s, int32_t mode, int32_t trace, double t_stop, int32_t flags) {
  if (!s || (mode != ORC_MODE_NAIVE && mode != ORC_MODE_FAST)) return ORC_EINVAL;
  if (flags & ~(ORC_FLAG_SETTLE_EVERY_EVENT | ORC_FLAG_F64_SHARES)) return ORC_EINVAL;
  if ((flags & ORC_FLAG_F64_SHARES) && mode != ORC_MODE_NAIVE) return ORC_EINVAL; /* dense argmin only */
  /* A run CONTINUES from the events kept so far (s->n_ev of them: all of an earlier run that stopped at a time, or
   * fewer after orc_rollback): the state after event K-1 is rebuilt from the throughput history, as PAPER.md L128
   * describes ("we know each flow's throughput at any given time, we can calculate the amount of data transferred
   * ... and consequently recover the simulator state").  The comparison modes and the trace are whole runs only. */
  if ((s->ran || s->n_ev > 0) && (flags || trace)) return ORC_ESTATE;
  int64_t F = s->F;
  const int64_t K = s->n_ev;
  int32_t L = s->n_links, rc = ORC_OK;
  ws_t w;
  memset(&w, 0, sizeof(w));
  int64_t *capq = (int64_t *)malloc(sizeof(int64_t) * L);
  int64_t *succ_off = (int64_t *)calloc(F + 1, sizeof(int64_t));
  int32_t *succ = (int32_t *)malloc(sizeof(int32_t) * (s->pred_off[F] + 1));
  int32_t *pred_cnt = (int32_t *)malloc(sizeof(int32_t) * (F + 1));
  uint8_t *state = (uint8_t *)calloc(F + 1, 1);
  double *t_act = (double *)malloc(sizeof(double) * (F + 1));
  double *rem = (double *)malloc(sizeof(double) * (F + 1));
  double *tc = (double *)malloc(sizeof(double) * (F + 1));
  int64_t *rq = (int64_t *)malloc(sizeof(int64_t) * (F + 1));
  int64_t *rq_cur = (int64_t *)malloc(sizeof(int64_t) * (F + 1)); /* rate in effect since t_last (R-LZ) */
  double *t_last = (double *)malloc(sizeof(double) * (F + 1));    /* time rem[] refers to (R-LZ)         */
  double *rate_d = (double *)malloc(sizeof(double) * (F + 1));     /* ORC_FLAG_F64_SHARES: binary64 rates       */
  double *rate_cur = (double *)malloc(sizeof(double) * (F + 1));   /* rate in effect since t_last, byte/s       */
  int32_t *act = (int32_t *)malloc(sizeof(int32_t) * (F + 1));
  int32_t *pend = (int32_t *)malloc(sizeof(int32_t) * (F + 1));
  int32_t *comp = (int32_t *)malloc(sizeof(int32_t) * (F + 1));
  if (s->F_res < F || !s->t_done) { /* results: kept across runs, extended for flows added since */
    void *a = realloc(s->t_done, sizeof(double) * (F + 1)), *b, *d;
    if (a) s->t_done = (double *)a;
    b = realloc(s->bneck, sizeof(int32_t) * (F + 1));
    if (b) s->bneck = (int32_t *)b;
    d = realloc(s->done_ev, sizeof(int64_t) * (F + 1));
    if (d) s->done_ev = (int64_t *)d;
    if (!a || !b || !d) { rc = ORC_ENOMEM; goto out; }
    for (int64_t f = s->F_res; f < F; f++) { s->t_done[f] = NAN; s->bneck[f] = -1; s->done_ev[f] = -1; }
    s->F_res = F;
  }
  if (!capq || !succ_off || !succ || !pred_cnt || !state || !t_act || !rem || !tc || !rq || !rq_cur || !t_last || !rate_d || !rate_cur || !act || !pend || !comp ||
      !s->t_done || !s->bneck || ws_init(&w, L)) {
    rc = ORC_ENOMEM;
    goto out;
  }
  for (int32_t l = 0; l < L; l++) {
    capq[l] = rate_to_q(s->cap[l]);
    if (capq[l] < F + 1) { rc = ORC_ERANGE; goto out; } /* every fair share stays >= 1 quantum */
  }
  if (K == 0) memset(s->work, 0, sizeof(s->work));
  /* successor lists = transpose of the pred lists */
  for (int64_t e = 0; e < s->pred_off[F]; e++) succ_off[s->pred[e] + 1]++;
  for (int64_t f = 0; f < F; f++) succ_off[f + 1] += succ_off[f];
  {
    int64_t *cur = (int64_t *)malloc(sizeof(int64_t) * (F + 1));
    if (!cur) { rc = ORC_ENOMEM; goto out; }
    memcpy(cur, succ_off, sizeof(int64_t) * (F + 1));
    for (int64_t f = 0; f < F; f++)
      for (int64_t e = s->pred_off[f]; e < s->pred_off[f + 1]; e++) succ[cur[s->pred[e]]++] = (int32_t)f;
    free(cur);
  }
  int32_t nA = 0, nP = 0, stopped = 0;
  int64_t n_done = 0;
  double now = K > 0 ? s->ev[K - 1].t : 0.0;
  /* ---- the state after event K-1 (K = 0: the initial state).  History records of iteration K and later are
   * dropped: the loop below writes them again.  A flow is DONE if it completed in an event < K; ACTIVE if it has a
   * record left -- the last one holds (time, rate, remaining bytes) of its current constant-throughput interval, and
   * its completion time is time + remaining / rate exactly as when the record was written; otherwise it waits for
   * its predecessors, or (all of them done) is PENDING with t_act = max(start, latest predecessor) + Lat. */
  {
    int64_t keep = 0;
    for (int64_t i = 0; i < s->n_h; i++)
      if (s->h_ev[i] < K) {
        s->h_flow[keep] = s->h_flow[i]; s->h_t[keep] = s->h_t[i]; s->h_rate[keep] = s->h_rate[i];
        s->h_rem[keep] = s->h_rem[i]; s->h_ev[keep] = s->h_ev[i]; s->h_rq[keep] = s->h_rq[i];
        keep++;
      }
    s->n_h = keep;
    for (int64_t f = 0; f < F; f++) {
      rq_cur[f] = -1;
      if (s->done_ev[f] >= K) { s->done_ev[f] = -1; s->t_done[f] = NAN; }
      if (s->done_ev[f] >= 0) { state[f] = DONE; n_done++; } else s->bneck[f] = -1;
    }
    for (int64_t i = 0; i < s->n_h; i++) { /* records are chronological: the last one of a flow wins */
      int32_t f = s->h_flow[i];
      if (state[f] == DONE) continue;
      t_last[f] = s->h_t[i];
      rate_cur[f] = s->h_rate[i];
      rq_cur[f] = s->h_rq[i];
      rem[f] = s->h_rem[i];
    }
    for (int64_t f = 0; f < F; f++) {
      if (state[f] == DONE) continue;
      if (rq_cur[f] >= 0) {
        state[f] = ACTIVE;
        double q = rem[f] / rate_cur[f];
        tc[f] = t_last[f] + q;
        act[nA++] = (int32_t)f;
        continue;
      }
      double latest = 0.0;
      pred_cnt[f] = 0;
      for (int64_t e = s->pred_off[f]; e < s->pred_off[f + 1]; e++) {
        int32_t p = s->pred[e];
        if (s->done_ev[p] >= 0) { if (s->t_done[p] > latest) latest = s->t_done[p]; }
        else pred_cnt[f]++;
      }
      if (pred_cnt[f] == 0) { /* released (or no preds): t_act = max(start, latest predecessor) + Lat -> PENDING */
        double st = s->start[f] > latest ? s->start[f] : latest;
        t_act[f] = st + s->Lat[f];
        state[f] = PENDING;
        pend[nP++] = (int32_t)f;
      }
    }
  }
  for (;;) {
    /* 1. activate every PENDING flow with t_act <= now */
    int32_t n_activated = 0, np2 = 0;
    for (int32_t i = 0; i < nP; i++) {
      int32_t f = pend[i];
      if (t_act[f] <= now) {
        rem[f] = s->bytes[f];
        rq_cur[f] = -1; /* no rate yet */
        state[f] = ACTIVE;
        act[nA++] = f;
        n_activated++;
      } else
        pend[np2++] = f;
    }
    nP = np2;
    /* 2. rates over all ACTIVE flows, from scratch (S5) */
    int32_t R = 0, fb = -1, lam = 0;
    if (flags & ORC_FLAG_F64_SHARES) {
      if (solve_maxmin_f64(&w, s->cap, nA, act, s->path_off, s->path, rate_d, s->bneck, &R, &fb, &lam)) {
        rc = ORC_ENOMEM;
        goto out;
      }
    } else if (solve_maxmin(&w, capq, nA, act, s->path_off, s->path, mode, rq, s->bneck, &R, &fb, &lam)) {
      rc = ORC_ENOMEM;
      goto out;
    }
    /* 3. settle + next time (reading R-LZ, PAPER.md L128 / L167: a flow's throughput is piecewise constant and
     *    its state is a function of its OWN rate changes).  A flow whose rate quanta did not change since its
     *    last rate change is not touched.  On a change at `now`: rem -= rate_old * (now - t_last) (mul, sub,
     *    clamp at 0), t_last = now, tc = now + rem / rate_new (div, then add).
     *    t_next = min(min tc, min pending t_act). */
    if (nA == 0 && nP == 0) break;
    double t_next = INFINITY;
    double ah = 0;
    for (int32_t i = 0; i < nA; i++) {
      int32_t f = act[i];
      double new_rate = (flags & ORC_FLAG_F64_SHARES) ? rate_d[f] : q_to_rate(rq[f]);
      int changed = (flags & ORC_FLAG_F64_SHARES) ? (rq_cur[f] < 0 || new_rate != rate_cur[f]) : (rq[f] != rq_cur[f]);
      if (changed) {
        if (s->n_h == s->h_cap) { /* history: the flow's throughput changes to new_rate at `now` */
          int64_t c = s->h_cap ? 2 * s->h_cap : 4096;
          void *a = realloc(s->h_flow, sizeof(int32_t) * c), *b, *d;
          if (!a) { rc = ORC_ENOMEM; goto out; }
          s->h_flow = (int32_t *)a;
          b = realloc(s->h_t, sizeof(double) * c);
          if (!b) { rc = ORC_ENOMEM; goto out; }
          s->h_t = (double *)b;
          d = realloc(s->h_rate, sizeof(double) * c);
          if (!d) { rc = ORC_ENOMEM; goto out; }
          s->h_rate = (double *)d;
          a = realloc(s->h_rem, sizeof(double) * c);
          if (!a) { rc = ORC_ENOMEM; goto out; }
          s->h_rem = (double *)a;
          b = realloc(s->h_ev, sizeof(int64_t) * c);
          if (!b) { rc = ORC_ENOMEM; goto out; }
          s->h_ev = (int64_t *)b;
          d = realloc(s->h_rq, sizeof(int64_t) * c);
          if (!d) { rc = ORC_ENOMEM; goto out; }
          s->h_rq = (int64_t *)d;
          s->h_cap = c;
        }
      }
      if (changed || ((flags & ORC_FLAG_SETTLE_EVERY_EVENT) && rq_cur[f] >= 0)) {
        if (rq_cur[f] >= 0) rem[f] = settle(rem[f], rate_cur[f], now - t_last[f]);
        t_last[f] = now;
        rq_cur[f] = (flags & ORC_FLAG_F64_SHARES) ? 0 : rq[f];
        rate_cur[f] = new_rate;
        double q = rem[f] / new_rate;
        tc[f] = now + q;
      }
      if (changed) { /* the record: (time, new rate, remaining bytes), written in iteration n_ev */
        s->h_flow[s->n_h] = f; s->h_t[s->n_h] = now; s->h_rate[s->n_h] = new_rate; s->h_rem[s->n_h] = rem[f];
        s->h_ev[s->n_h] = s->n_ev; s->h_rq[s->n_h] = rq_cur[f]; s->n_h++;
      }
      if (tc[f] < t_next) t_next = tc[f];
      ah += (double)(s->path_off[f + 1] - s->path_off[f]);
    }
    for (int32_t i = 0; i < nP; i++)
      if (t_act[pend[i]] < t_next) t_next = t_act[pend[i]];
    if (t_next > t_stop) { stopped = 1; break; } /* the next event lies beyond the requested time */
    /* 4. advance: flows whose completion time is bit-equal to t_next complete; nobody else changes */
    int32_t nC = 0, na2 = 0;
    for (int32_t i = 0; i < nA; i++) {
      int32_t f = act[i];
      if (trace) {
        if (s->n_tr == s->tr_cap) {
          int64_t c = s->tr_cap ? 2 * s->tr_cap : 4096;
          void *q = realloc(s->tr, sizeof(trace_row) * c);
          if (!q) { rc = ORC_ENOMEM; goto out; }
          s->tr = (trace_row *)q; s->tr_cap = c;
        }
        trace_row *r = &s->tr[s->n_tr++];
        r->ev = s->n_ev; r->flow = f; r->rate = rate_cur[f]; r->t0 = now; r->t1 = t_next;
      }
      if (tc[f] == t_next) { /* bit-equal absolute time: completes */
        s->t_done[f] = t_next;
        s->done_ev[f] = s->n_ev;
        state[f] = DONE;
        comp[nC++] = f;
      } else {
        act[na2++] = f;
      }
    }
    s->work[0] += nA; s->work[1] += ah; s->work[2] += R; s->work[3] += (double)lam * R; s->work[4] += lam;
    s->work[5] += nC; s->work[6] += 1;
    nA = na2;
    n_done += nC;
    now = t_next;
    /* 5. release successors of completed flows (ascending id: comp[] is in act[] order; order is immaterial,
     *    every update is a counter decrement or a function of `now` only) */
    for (int32_t i = 0; i < nC; i++)
      for (int64_t e = succ_off[comp[i]]; e < succ_off[comp[i] + 1]; e++) {
        int32_t g = succ[e];
        if (--pred_cnt[g] == 0) {
          double st = s->start[g] > now ? s->start[g] : now;
          t_act[g] = st + s->Lat[g];
          state[g] = PENDING;
          pend[nP++] = g;
        }
      }
    /* 6. log */
    if (s->n_ev == s->ev_cap) {
      int64_t c = s->ev_cap ? 2 * s->ev_cap : 1024;
      void *q = realloc(s->ev, sizeof(orc_event) * c);
      if (!q) { rc = ORC_ENOMEM; goto out; }
      s->ev = (orc_event *)q; s->ev_cap = c;
    }
    orc_event *e = &s->ev[s->n_ev++];
    e->t = t_next; e->n_completed = nC; e->n_activated = n_activated; e->n_rounds = R; e->first_bneck = fb;
  }
  if (stopped) { /* unfinished flows report no bottleneck */
    for (int64_t f = 0; f < F; f++)
      if (state[f] != DONE) s->bneck[f] = -1;
  } else if (n_done < F) rc = ORC_ECYCLE; /* WAITING flows left with nothing active or pending */
  s->ran = 1;
out:
  free(capq); free(succ_off); free(succ); free(pred_cnt); free(state); free(t_act); free(rem); free(tc); free(rq); free(rq_cur); free(t_last);
  free(rate_d); free(rate_cur); free(act); free(pend); free(comp);
  ws_free(&w);
  return rc;
}

/* ------------------------------------------------------------------ S6: outputs */
int32_t orc_num_flows(const orc_sim *s, int64_t *out) { if (!s || !out) return ORC_EINVAL; *out = s->F; return ORC_OK; }
int32_t orc_get_completion_times(const orc_sim *s, double *out, int64_t n) {
  if (!s || !out || n != s->F) return ORC_EINVAL;
  if (!s->t_done) return ORC_ESTATE;
  memcpy(out, s->t_done, sizeof(double) * n);
  return ORC_OK;
}
int32_t orc_get_bottlenecks(const orc_sim *s, int32_t *out, int64_t n) {
  if (!s || !out || n != s->F) return ORC_EINVAL;
  if (!s->bneck) return ORC_ESTATE;
  memcpy(out, s->bneck, sizeof(int32_t) * n);
  return ORC_OK;
}
int32_t orc_num_collectives(const orc_sim *s, int32_t *out) { if (!s || !out) return ORC_EINVAL; *out = s->n_coll; return ORC_OK; }
int32_t orc_get_collective_times(const orc_sim *s, double *out, int32_t n) {
  if (!s || !out || n != s->n_coll) return ORC_EINVAL;
  if (!s->t_done) return ORC_ESTATE;
  for (int32_t c = 0; c < n; c++) { /* O5: max t_done over the collective's flows */
    double m = -INFINITY;
    int open_flows = 0; /* after orc_run_until: a collective with unfinished flows has no finish time yet */
    for (int32_t f = s->coll[c].first_flow; f < s->coll[c].first_flow + s->coll[c].n_flows; f++) {
      if (s->t_done[f] != s->t_done[f]) open_flows = 1;
      if (s->t_done[f] > m) m = s->t_done[f];
    }
    out[c] = open_flows ? NAN : m;
  }
  return ORC_OK;
}
int32_t orc_num_events(const orc_sim *s, int64_t *out) { if (!s || !out) return ORC_EINVAL; *out = s->n_ev; return ORC_OK; }
int32_t orc_get_event_log(const orc_sim *s, orc_event *out, int64_t cap, int64_t *n) {
  if (!s || !n) return ORC_EINVAL;
  *n = s->n_ev;
  if (out) memcpy(out, s->ev, sizeof(orc_event) * (cap < s->n_ev ? cap : s->n_ev));
  return ORC_OK;
}
int32_t orc_num_path_entries(const orc_sim *s, int64_t *out) { if (!s || !out) return ORC_EINVAL; *out = s->path_off[s->F]; return ORC_OK; }
int32_t orc_get_paths(const orc_sim *s, int64_t *off, int32_t *links, int64_t cap) {
  if (!s || !off || !links || cap < s->path_off[s->F]) return ORC_EINVAL;
  memcpy(off, s->path_off, sizeof(int64_t) * (s->F + 1));
  memcpy(links, s->path, sizeof(int32_t) * s->path_off[s->F]);
  return ORC_OK;
}
int32_t orc_get_flow_endpoints(const orc_sim *s, int32_t *src, int32_t *dst, double *bytes, double *lat, int64_t n) {
  if (!s || n != s->F) return ORC_EINVAL;
  if (src) memcpy(src, s->src, sizeof(int32_t) * n);
  if (dst) memcpy(dst, s->dst, sizeof(int32_t) * n);
  if (bytes) memcpy(bytes, s->bytes, sizeof(double) * n);
  if (lat) memcpy(lat, s->Lat, sizeof(double) * n);
  return ORC_OK;
}
int32_t orc_get_preds(const orc_sim *s, int64_t *off, int32_t *preds, int64_t cap, int64_t *n_entries) {
  if (!s || !n_entries) return ORC_EINVAL;
  *n_entries = s->pred_off[s->F];
  if (off) memcpy(off, s->pred_off, sizeof(int64_t) * (s->F + 1));
  if (preds) {
    if (cap < *n_entries) return ORC_EINVAL;
    memcpy(preds, s->pred, sizeof(int32_t) * *n_entries);
  }
  return ORC_OK;
}
int32_t orc_get_work_counters(const orc_sim *s, double *out7) {
  if (!s || !out7) return ORC_EINVAL;
  memcpy(out7, s->work, sizeof(s->work));
  return ORC_OK;
}
int32_t orc_history_size(const orc_sim *s, int64_t *n) { if (!s || !n) return ORC_EINVAL; *n = s->n_h; return ORC_OK; }
int32_t orc_get_history(const orc_sim *s, int32_t *flow, double *t, double *rate, int64_t cap) {
  if (!s || cap < s->n_h) return ORC_EINVAL;
  for (int64_t i = 0; i < s->n_h; i++) { flow[i] = s->h_flow[i]; t[i] = s->h_t[i]; rate[i] = s->h_rate[i]; }
  return ORC_OK;
}
int32_t orc_trace_size(const orc_sim *s, int64_t *n) { if (!s || !n) return ORC_EINVAL; *n = s->n_tr; return ORC_OK; }
int32_t orc_get_trace(const orc_sim *s, int64_t *ev, int32_t *flow, double *rate, double *t0, double *t1, int64_t cap) {
  if (!s || cap < s->n_tr) return ORC_EINVAL;
  for (int64_t i = 0; i < s->n_tr; i++) {
    if (ev) ev[i] = s->tr[i].ev;
    if (flow) flow[i] = s->tr[i].flow;
    if (rate) rate[i] = s->tr[i].rate;
    if (t0) t0[i] = s->tr[i].t0;
    if (t1) t1[i] = s->tr[i].t1;
  }
  return ORC_OK;
}
