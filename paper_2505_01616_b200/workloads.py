"""Seeded synthetic input generators (BASELINE.json configs 0-4 and scaled-down variants).

This module holds NONE of the method's arithmetic: it only draws the inputs (topology descriptor, per-instance
link capacities, collectives, raw flows) that are then handed, as plain arrays, to BOTH the CUDA library and the
CPU oracle.  It imports neither.  The recipe is stated in DESIGN.md ("Input recipe").  The paper evaluates on
real training jobs (Table 1), not on a public network benchmark; these inputs stand in for
the *shape* of that traffic (TP/DP ring collectives, L104/L248; MoE all-to-all, L316).
"""
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

TOPO_SINGLE, TOPO_LEAF_SPINE, TOPO_FAT_TREE = 0, 1, 2
ALLREDUCE_RING, ALLGATHER_RING, REDUCESCATTER_RING, ALLTOALL = 0, 1, 2, 3
BROADCAST_CHAIN, REDUCE_CHAIN, ALLREDUCE_TREE = 4, 5, 6

MiB = float(2 ** 20)
GiB = float(2 ** 30)
KiB = float(2 ** 10)


def gbps(x):
    """x Gb/s -> byte/s."""
    return x * 1e9 / 8.0


def topo_desc(kind, n_hosts, gpus_per_host, nvlink_Bps=450e9, nic_Bps=50e9, fabric_Bps=50e9, hop_latency_s=1e-6,
              n_leaves=0, n_spines=0, uplinks_per_leaf_spine=0, k=0, agg_uplinks=0, compute_lanes=0):
    return dict(kind=kind, n_hosts=n_hosts, gpus_per_host=gpus_per_host, nvlink_Bps=nvlink_Bps, nic_Bps=nic_Bps,
                fabric_Bps=fabric_Bps, hop_latency_s=hop_latency_s, n_leaves=n_leaves, n_spines=n_spines,
                uplinks_per_leaf_spine=uplinks_per_leaf_spine, k=k, agg_uplinks=agg_uplinks,
                compute_lanes=compute_lanes)


def graph_desc(n_gpus, n_nodes, link_from, link_to, cap_Bps, latency_s, compute_lanes=0):
    """User-supplied topology (NEXT-4): nodes 0..n_gpus-1 are GPUs, the rest switches; link i is the directed edge
    link_from[i] -> link_to[i]."""
    return dict(graph=dict(n_gpus=n_gpus, n_nodes=n_nodes, link_from=np.asarray(link_from, np.int32),
                           link_to=np.asarray(link_to, np.int32), cap_Bps=np.asarray(cap_Bps, np.float64),
                           latency_s=np.asarray(latency_s, np.float64), compute_lanes=compute_lanes),
                n_hosts=n_gpus, gpus_per_host=1, compute_lanes=compute_lanes, nvlink_Bps=0.0)


@dataclass
class Coll:
    kind: int
    ranks: np.ndarray
    nbytes: float
    start: float = 0.0
    after: tuple = ()
    chunks: int = 1          # pipeline chunks of the chain / tree kinds
    after_flows: tuple = ()  # flow / span ids its initial flows additionally wait for (per rank)


@dataclass
class Spans:
    """Compute spans (NEXT-2): fixed-duration DAG nodes on a compute lane of a GPU."""
    gpu: np.ndarray
    duration: np.ndarray
    lane: Optional[np.ndarray] = None
    start: Optional[np.ndarray] = None
    dep_off: Optional[np.ndarray] = None
    dep_ids: Optional[np.ndarray] = None


@dataclass
class RawFlows:
    src: np.ndarray
    dst: np.ndarray
    nbytes: np.ndarray
    start: Optional[np.ndarray] = None
    dep_off: Optional[np.ndarray] = None
    dep_ids: Optional[np.ndarray] = None
    conn_id: Optional[np.ndarray] = None


@dataclass
class Instance:
    seed: int
    ops: list = field(default_factory=list)          # Coll | RawFlows, in submission order
    cap_pairs_Gbps: Optional[np.ndarray] = None      # cfg3: one draw per physical NIC/fabric link

    def capacities(self, desc, n_links):
        """Per-directed-link capacity array, or None for the descriptor's defaults.  Uses only the numbering
        convention of DESIGN.md S1: links [0,2G) NVLink; from 2G on, physical link p = directed pair (2G+2p, 2G+2p+1)."""
        if self.cap_pairs_Gbps is None:
            return None
        G = desc["n_hosts"] * desc["gpus_per_host"]
        n_net = n_links - G * desc.get("compute_lanes", 0)       # compute engine links follow the network links
        cap = np.full(n_links, desc["nvlink_Bps"], dtype=np.float64)
        pairs = (n_net - 2 * G) // 2
        assert len(self.cap_pairs_Gbps) == pairs
        cap[2 * G:n_net:2] = gbps(self.cap_pairs_Gbps)
        cap[2 * G + 1:n_net:2] = gbps(self.cap_pairs_Gbps)
        cap[n_net:] = 2.0 ** 32                                   # work units / s of a compute lane
        return cap

    @property
    def n_collectives(self):
        n = sum(1 for o in self.ops if isinstance(o, Coll))
        return n if n else 1      # a raw-flow instance counts as one all-to-all-equivalent (cfg4)


def capacity_matrix(desc, insts, n_links):
    """Instance.capacities of every instance as one [len(insts)][n_links] array (same numbering convention), or None
    unless all of them override the capacities."""
    if not insts or any(x.cap_pairs_Gbps is None for x in insts):
        return None
    G = desc["n_hosts"] * desc["gpus_per_host"]
    n_net = n_links - G * desc.get("compute_lanes", 0)
    pairs = (n_net - 2 * G) // 2
    p = np.stack([np.asarray(x.cap_pairs_Gbps, dtype=np.float64) for x in insts])
    assert p.shape == (len(insts), pairs)
    cap = np.full((len(insts), n_links), desc["nvlink_Bps"], dtype=np.float64)
    cap[:, 2 * G:n_net:2] = gbps(p)
    cap[:, 2 * G + 1:n_net:2] = gbps(p)
    cap[:, n_net:] = 2.0 ** 32
    return cap


@dataclass
class Workload:
    name: str
    desc: dict
    base_seed: int
    instances: List[Instance]
    uniform_ops: bool = False   # every instance has the same collectives (kind, ranks, after); only sizes / starts differ

    @property
    def batch(self):
        return len(self.instances)


def n_flows_of(op):
    if isinstance(op, RawFlows):
        return len(op.src)
    if isinstance(op, Spans):
        return len(op.gpu)
    N = len(op.ranks)
    return {ALLREDUCE_RING: 2 * (N - 1) * N, ALLGATHER_RING: (N - 1) * N, REDUCESCATTER_RING: (N - 1) * N,
            ALLTOALL: N * (N - 1), BROADCAST_CHAIN: op.chunks * (N - 1), REDUCE_CHAIN: op.chunks * (N - 1),
            ALLREDUCE_TREE: op.chunks * 2 * (N - 1)}[op.kind]


def _rng(cfg, instance):
    return np.random.Generator(np.random.PCG64([0x2505_01616, cfg, instance]))


def _loguniform(rng, lo, hi, size=None):
    """exp(U(ln lo, ln hi)), floored to whole bytes."""
    return np.floor(np.exp(rng.uniform(np.log(lo), np.log(hi), size)))


def batched_sizes(w, first, count):
    """For a workload whose instances have the same collectives (uniform_ops): the per-instance sizes and start times of
    collective k as host arrays nbytes[k][count], start[k][count] -- the form phs_add_collective_batch takes.  Built
    once per (first, count) and kept on the workload (input preparation, like the generator itself)."""
    cache = w.__dict__.setdefault("_batched", {})
    if (first, count) not in cache:
        insts = w.instances[first:first + count]
        n_ops = len(insts[0].ops)
        nb = np.array([[op.nbytes for op in x.ops] for x in insts], np.float64).T.copy()
        st = np.array([[op.start for op in x.ops] for x in insts], np.float64).T.copy()
        assert nb.shape == (n_ops, count)
        cache[(first, count)] = (nb, st)
    return cache[(first, count)]


def apply(inst: Instance, add_collective, add_flows, add_spans=None):
    """Replay an instance's ops through callables with the signatures
    add_collective(kind, ranks, nbytes, start, after[, chunks[, after_flows]]) -> id ;
    add_flows(src, dst, nbytes, start, dep_off, dep_ids, conn_id) ; add_spans(gpu, duration, lane, start, dep_off, dep_ids)."""
    for op in inst.ops:
        if isinstance(op, Spans):
            add_spans(op.gpu, op.duration, op.lane, op.start, op.dep_off, op.dep_ids)
        elif isinstance(op, Coll):
            if len(op.after_flows):
                add_collective(op.kind, op.ranks, op.nbytes, op.start, op.after, op.chunks, op.after_flows)
            elif op.chunks == 1:
                add_collective(op.kind, op.ranks, op.nbytes, op.start, op.after)
            else:
                add_collective(op.kind, op.ranks, op.nbytes, op.start, op.after, op.chunks)
        else:
            add_flows(op.src, op.dst, op.nbytes, op.start, op.dep_off, op.dep_ids, op.conn_id)


# ---------------------------------------------------------------------------------------------- cfg0
def cfg0():
    """16 GPUs (2x8) on one switch; one ring all-reduce of 64 MiB over ranks 0..15; batch 1; seed 0."""
    d = topo_desc(TOPO_SINGLE, 2, 8)
    inst = Instance(seed=0, ops=[Coll(ALLREDUCE_RING, np.arange(16, dtype=np.int32), 64 * MiB)])
    return Workload("cfg0", d, 0, [inst])


# ---------------------------------------------------------------------------------------------- cfg1
def cfg1(batch=64, n_hosts=16, gph=8, n_leaves=4, n_spines=2):
    """Leaf-spine; per instance: one TP ring all-reduce per host + one DP ring all-reduce per local rank, all at
    t=0.  Instance 0: 16 MiB / 1 GiB; instances >=1: every collective log-uniform in [1 MiB, 4 GiB]."""
    d = topo_desc(TOPO_LEAF_SPINE, n_hosts, gph, fabric_Bps=gbps(400.0), n_leaves=n_leaves, n_spines=n_spines,
                  uplinks_per_leaf_spine=1)
    insts = []
    for i in range(batch):
        rng = _rng(1, i)
        ops = []
        for h in range(n_hosts):
            sz = 16 * MiB if i == 0 else float(_loguniform(rng, 1 * MiB, 4 * GiB))
            ops.append(Coll(ALLREDUCE_RING, np.arange(h * gph, (h + 1) * gph, dtype=np.int32), sz))
        for j in range(gph):
            sz = 1 * GiB if i == 0 else float(_loguniform(rng, 1 * MiB, 4 * GiB))
            ops.append(Coll(ALLREDUCE_RING, np.arange(j, n_hosts * gph, gph, dtype=np.int32), sz))
        insts.append(Instance(seed=i, ops=ops))
    return Workload("cfg1", d, 0, insts, uniform_ops=True)


# ---------------------------------------------------------------------------------------------- cfg2
def cfg2(k=16, agg_uplinks=4, dp_colls=(ALLREDUCE_RING, ALLREDUCE_RING, ALLGATHER_RING, ALLGATHER_RING,
                                        REDUCESCATTER_RING, REDUCESCATTER_RING),
         tp_colls=(ALLREDUCE_RING, ALLGATHER_RING, REDUCESCATTER_RING)):
    """k-ary 3-tier fat tree (2:1 at the aggregation tier for agg_uplinks = k/4); TP groups = hosts, DP groups =
    local ranks; bytes log-uniform [64 KiB, 1 GiB]; start times uniform [0, 10 ms]; one instance, seed 0."""
    gph, n_hosts = k // 2, k * (k // 2)
    d = topo_desc(TOPO_FAT_TREE, n_hosts, gph, fabric_Bps=gbps(400.0), k=k, agg_uplinks=agg_uplinks)
    rng = _rng(2, 0)
    ops = []
    for j in range(gph):
        ranks = np.arange(j, n_hosts * gph, gph, dtype=np.int32)
        for kind in dp_colls:
            ops.append(Coll(kind, ranks, float(_loguniform(rng, 64 * KiB, 1 * GiB)), float(rng.uniform(0.0, 10e-3))))
    for h in range(n_hosts):
        ranks = np.arange(h * gph, (h + 1) * gph, dtype=np.int32)
        for kind in tp_colls:
            ops.append(Coll(kind, ranks, float(_loguniform(rng, 64 * KiB, 1 * GiB)), float(rng.uniform(0.0, 10e-3))))
    return Workload("cfg2", d, 0, [Instance(seed=0, ops=ops)])


# ---------------------------------------------------------------------------------------------- cfg3
def cfg3(batch=4096, n_hosts=8, gph=8, n_leaves=2, n_spines=2, layers=4, buckets=4):
    """Parameter sweep: per instance, NIC and fabric capacities U[100,800] Gb/s per physical link; one training
    step = `layers` TP layers (one ring all-reduce per host, chained per host with `after`) + `buckets` gradient
    buckets (one DP ring all-reduce per local rank, chained); sizes log-uniform [1 MiB, 1 GiB]."""
    d = topo_desc(TOPO_LEAF_SPINE, n_hosts, gph, fabric_Bps=gbps(400.0), n_leaves=n_leaves, n_spines=n_spines,
                  uplinks_per_leaf_spine=1)
    G = n_hosts * gph
    pairs = G + n_leaves * n_spines
    insts = []
    for i in range(batch):
        rng = _rng(3, i)
        caps = rng.uniform(100.0, 800.0, pairs)
        ops = []
        for layer in range(layers):
            for h in range(n_hosts):
                after = () if layer == 0 else ((layer - 1) * n_hosts + h,)
                ops.append(Coll(ALLREDUCE_RING, np.arange(h * gph, (h + 1) * gph, dtype=np.int32),
                                float(_loguniform(rng, 1 * MiB, 1 * GiB)), 0.0, after))
        base = layers * n_hosts
        for b in range(buckets):
            for j in range(gph):
                after = () if b == 0 else (base + (b - 1) * gph + j,)
                ops.append(Coll(ALLREDUCE_RING, np.arange(j, G, gph, dtype=np.int32),
                                float(_loguniform(rng, 1 * MiB, 1 * GiB)), 0.0, after))
        insts.append(Instance(seed=i, ops=ops, cap_pairs_Gbps=caps))
    return Workload("cfg3", d, 0, insts, uniform_ops=True)


# ---------------------------------------------------------------------------------------------- cfg4
def cfg4(batch=8, n_hosts=32, gph=8, n_leaves=8, n_spines=8, mean_bytes=4 * MiB, zipf_a=1.2):
    """MoE all-to-all stress: raw flows for every ordered GPU pair, all at t=0; destination popularity Zipf(a) over
    a seeded permutation pi: bytes(s->d) = (G-1)*mean * pi(d)^-a / sum_{d'!=s} pi(d')^-a * U[0.75,1.25), floored
    to whole bytes (>= 1)."""
    d = topo_desc(TOPO_LEAF_SPINE, n_hosts, gph, fabric_Bps=gbps(400.0), n_leaves=n_leaves, n_spines=n_spines,
                  uplinks_per_leaf_spine=1)
    G = n_hosts * gph
    insts = []
    for i in range(batch):
        rng = _rng(4, i)
        pi = rng.permutation(G) + 1
        w = pi.astype(np.float64) ** (-zipf_a)
        src = np.repeat(np.arange(G, dtype=np.int32), G)
        dst = np.tile(np.arange(G, dtype=np.int32), G)
        keep = src != dst
        src, dst = src[keep], dst[keep]
        denom = w.sum() - w                                   # per source: sum over d' != s
        nbytes = (G - 1) * mean_bytes * w[dst] / denom[src] * rng.uniform(0.75, 1.25, len(src))
        nbytes = np.maximum(np.floor(nbytes), 1.0)
        insts.append(Instance(seed=i, ops=[RawFlows(src, dst, nbytes)]))
    return Workload("cfg4", d, 0, insts)


# ---------------------------------------------------------------------------------------------- training step
def train_step(batch=4, n_hosts=8, gph=8, n_leaves=2, n_spines=2, layers=4, buckets=4):
    """cfg3's sweep with the compute of the step in the DAG (NEXT-2, PAPER.md L84 / L206): per layer one compute span
    per GPU (U[20, 200] us; it waits for what that GPU sent and received in the previous layer's tensor-parallel
    all-reduce), then the layer's TP all-reduce per host (a rank starts when its span is done); after the last layer
    the gradient buckets, one DP all-reduce per local rank each, chained, the first behind the last layer's spans."""
    d = topo_desc(TOPO_LEAF_SPINE, n_hosts, gph, fabric_Bps=gbps(400.0), n_leaves=n_leaves, n_spines=n_spines,
                  uplinks_per_leaf_spine=1, compute_lanes=1)
    G = n_hosts * gph
    pairs = G + n_leaves * n_spines
    tp_flows = 2 * (gph - 1) * gph
    insts = []
    for i in range(batch):
        rng = _rng(5, i)
        caps = rng.uniform(100.0, 800.0, pairs)
        ops, nf, nc = [], 0, 0
        prev_tp_first = None                       # first flow id of the previous layer's TP all-reduce, per host
        span_first = 0
        for layer in range(layers):
            dep_off, dep_ids = [0], []
            for g in range(G):
                if prev_tp_first is not None:
                    h, pos = divmod(g, gph)
                    last = prev_tp_first[h] + (2 * (gph - 1) - 1) * gph
                    dep_ids += [last + pos, last + (pos - 1) % gph]
                dep_off.append(len(dep_ids))
            span_first = nf
            ops.append(Spans(np.arange(G, dtype=np.int32), rng.uniform(20e-6, 200e-6, G), None, None,
                             np.array(dep_off, np.int64), np.array(dep_ids, np.int64)))
            nf += G
            prev_tp_first = []
            for h in range(n_hosts):
                prev_tp_first.append(nf)
                ops.append(Coll(ALLREDUCE_RING, np.arange(h * gph, (h + 1) * gph, dtype=np.int32),
                                float(_loguniform(rng, 1 * MiB, 64 * MiB)), 0.0, (), 1,
                                tuple(range(span_first + h * gph, span_first + (h + 1) * gph))))
                nf += tp_flows
                nc += 1
        base = nc
        for b in range(buckets):
            for j in range(gph):
                after = () if b == 0 else (base + (b - 1) * gph + j,)
                after_flows = tuple(range(span_first + j, span_first + G, gph)) if b == 0 else ()
                ops.append(Coll(ALLREDUCE_RING, np.arange(j, G, gph, dtype=np.int32),
                                float(_loguniform(rng, 1 * MiB, 256 * MiB)), 0.0, after, 1, after_flows))
                nc += 1
        insts.append(Instance(seed=i, ops=ops, cap_pairs_Gbps=caps))
    return Workload("train_step", d, 0, insts)


def graph_fabric(batch=2, n_gpus=16, gpus_per_leaf=4, n_spines=3, seed0=0):
    """A user-supplied topology (NEXT-4): GPUs on leaf switches, every leaf wired to every spine, per-link capacities
    U[100, 800] Gb/s and latencies U[0.5, 2] us (both directions drawn separately), one compute lane per GPU; on it a
    mix of ring, tree and chain collectives with compute spans."""
    n_leaves = n_gpus // gpus_per_leaf
    rng = _rng(6, seed0)
    lf, lt = [], []
    for g in range(n_gpus):
        leaf = n_gpus + g // gpus_per_leaf
        lf += [g, leaf]; lt += [leaf, g]
    for leaf in range(n_leaves):
        for sp in range(n_spines):
            a, b = n_gpus + leaf, n_gpus + n_leaves + sp
            lf += [a, b]; lt += [b, a]
    n = len(lf)
    d = graph_desc(n_gpus, n_gpus + n_leaves + n_spines, lf, lt, gbps(rng.uniform(100.0, 800.0, n)),
                   rng.uniform(0.5e-6, 2e-6, n), compute_lanes=1)
    insts = []
    for i in range(batch):
        r = _rng(6, 100 + i)
        perm = r.permutation(n_gpus).astype(np.int32)
        ops = [Spans(np.arange(n_gpus, dtype=np.int32), r.uniform(10e-6, 80e-6, n_gpus)),
               Coll(ALLREDUCE_RING, perm[:8], float(_loguniform(r, 1 * MiB, 64 * MiB)), 0.0, (), 1, tuple(range(n_gpus))),
               Coll(ALLREDUCE_TREE, perm[4:15], float(_loguniform(r, 1 * MiB, 16 * MiB)), 1e-5, (), 3),
               Coll(BROADCAST_CHAIN, perm[8:], float(_loguniform(r, 1 * MiB, 16 * MiB)), 0.0, (0,), 4),
               Coll(ALLTOALL, perm[2:10], float(_loguniform(r, 1 * MiB, 8 * MiB)), 2e-5, (1,))]
        insts.append(Instance(seed=i, ops=ops))
    return Workload("graph_fabric", d, 7, insts)


def by_name(name, **kw):
    return {"cfg0": cfg0, "cfg1": cfg1, "cfg2": cfg2, "cfg3": cfg3, "cfg4": cfg4}[name](**kw)
