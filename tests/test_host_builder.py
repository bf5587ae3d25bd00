"""CPU-side tests of the library: the C-ABI loads and exports every symbol of include/phs.h; the host builder's
integer artefacts (ECMP paths, dependency DAG, flow table) equal the oracle's exactly; error behaviour; and the
product path fails loudly (no CPU fallback) when no CUDA device is usable."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import orc
from paper_2505_01616_b200 import binding as B
from paper_2505_01616_b200 import workloads as W
from util import oracle_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "phs.h")).read()
    declared = set(re.findall(r"\b(phs_[a-z_]+)\s*\(", hdr))
    declared -= {"phs_sim", "phs_status"}
    assert declared == set(B.SYMBOLS), declared ^ set(B.SYMBOLS)
    lib = B.lib()
    for name in declared:
        assert hasattr(lib, name), name


def _compare_tables(w, first=0, count=None):
    count = w.batch if count is None else count
    sim = B.Sim.from_workload(w, instances=(first, count))
    for i in range(count):
        o = oracle_build(w.desc, w.instances[first + i], base_seed=w.base_seed)
        off, links = sim.paths(i)
        ooff, olinks = o.paths()
        assert np.array_equal(off, ooff) and np.array_equal(links, olinks)
        # a3, the transpose (link -> flows, ascending flow id), against the transpose of the ORACLE's paths
        loff, lflows = sim.link_flows(i)
        flow_of_entry = np.repeat(np.arange(len(ooff) - 1, dtype=np.int32), np.diff(ooff))
        order = np.argsort(olinks, kind="stable")
        assert np.array_equal(lflows, flow_of_entry[order])
        assert np.array_equal(loff, np.concatenate([[0], np.cumsum(np.bincount(olinks, minlength=len(loff) - 1))]))
        poff, pr = sim.preds(i)
        opoff, opr = o.preds()
        assert np.array_equal(poff, opoff) and np.array_equal(pr, opr)
        for a, b in zip(sim.flows(i), o.flows()):
            assert np.array_equal(a, b)
        assert B.phs_num_collectives(sim.h, i) == o.num_collectives
        assert np.array_equal(B.phs_get_link_capacities(sim.h, i), o.link_capacities())
    sim.close()


@pytest.mark.parametrize("wl", [
    lambda: W.cfg0(),
    lambda: W.cfg1(batch=3),
    lambda: W.cfg2(k=8, agg_uplinks=2),
    lambda: W.cfg3(batch=3),
    lambda: W.cfg4(batch=2, n_hosts=8, gph=4, n_leaves=4, n_spines=2),
])
def test_paths_dag_and_flow_table_equal_the_oracle(wl):
    _compare_tables(wl())


def test_full_size_tables_equal_the_oracle():
    _compare_tables(W.cfg2())                       # 1,069,056 flows, 6-hop fat-tree paths
    _compare_tables(W.cfg4(batch=2), first=1, count=1)
    _compare_tables(W.cfg3(batch=130), first=128, count=2)   # seed = instance survives sub-batching


def test_after_and_alltoall_dag_equal_the_oracle():
    d = W.topo_desc(W.TOPO_LEAF_SPINE, 4, 4, n_leaves=2, n_spines=2, uplinks_per_leaf_spine=2)
    ops = [W.Coll(W.ALLTOALL, np.arange(0, 16, 2, dtype=np.int32), 8e6),
           W.Coll(W.ALLREDUCE_RING, np.array([2, 3, 4, 9, 8], np.int32), 5e6, 1e-4, (0,)),
           W.Coll(W.ALLTOALL, np.array([8, 4, 1], np.int32), 3e6, 0.0, (0, 1)),
           W.RawFlows(np.array([0, 1, 2], np.int32), np.array([5, 6, 7], np.int32), np.array([1e5, 2e5, 3e5]),
                      dep_off=np.array([0, 0, 1, 3]), dep_ids=np.array([0, 0, 1]), conn_id=np.array([7, 7, 9], np.int32)),
           W.Coll(W.REDUCESCATTER_RING, np.array([15, 0, 7], np.int32), 6e6, 0.0, (2,))]
    _compare_tables(W.Workload("mixed", d, 5, [W.Instance(seed=0, ops=ops), W.Instance(seed=1, ops=ops)]))


def test_chain_and_tree_collectives_equal_the_oracle():
    """NEXT-3 kinds: flows, routes and DAG (incl. `after` edges in both directions with every other kind) built by the
    library equal the oracle's, which is pinned against hand-written lists and closed forms (test_oracle_pins.py)."""
    d = W.topo_desc(W.TOPO_FAT_TREE, 8, 2, k=4, agg_uplinks=1)
    rng = np.random.default_rng(3)
    insts = []
    for i in range(3):
        perm = rng.permutation(16).astype(np.int32)
        ops = [W.Coll(W.BROADCAST_CHAIN, perm[:7], 8e6, 0.0, (), 5),
               W.Coll(W.ALLREDUCE_TREE, perm[3:14], 6e6, 1e-5, (), 3),
               W.Coll(W.REDUCE_CHAIN, perm[5:12], 4e6, 0.0, (0, 1), 4),
               W.Coll(W.ALLREDUCE_RING, perm[:6], 16e6, 0.0, (1, 2)),
               W.Coll(W.ALLTOALL, perm[8:14], 3e6, 2e-5, (2,)),
               W.Coll(W.ALLREDUCE_TREE, perm[1:9], 2e6, 0.0, (3, 4), 1),
               W.Coll(W.ALLREDUCE_TREE, np.array([perm[0], perm[15]], np.int32), 2e6, 0.0, (5,), 2),
               W.Coll(W.BROADCAST_CHAIN, perm[9:16], 5e6, 0.0, (5, 4, 6), 2),
               W.Coll(W.ALLGATHER_RING, perm[2:10], 5e6, 0.0, (7, 0))]
        insts.append(W.Instance(seed=i, ops=ops))
    _compare_tables(W.Workload("next3", d, 4, insts))
    sim = B.Sim(d, batch=1)
    for bad in (dict(kind=B.ALLREDUCE_RING, chunks=2), dict(kind=B.ALLREDUCE_TREE, chunks=0), dict(kind=7, chunks=1)):
        with pytest.raises(B.PhsError) as e:
            B.phs_add_collective(sim.h, 0, bad["kind"], [0, 1, 2], 1e6, chunks=bad["chunks"]) if bad["chunks"] != 1 else \
                B.phs_add_collective(sim.h, 0, bad["kind"], [0, 1, 2], 1e6)
        assert e.value.code == B.PHS_EINVAL
    sim.close()


def test_compute_spans_and_flow_level_after_edges_equal_the_oracle():
    """NEXT-2: a training step with compute spans in the DAG (spans behind collectives, collectives behind spans)."""
    _compare_tables(W.train_step(batch=3, n_hosts=4, gph=4, layers=3, buckets=2))
    d = W.topo_desc(W.TOPO_SINGLE, 2, 4)
    sim = B.Sim(d, batch=1)
    with pytest.raises(B.PhsError) as e:
        B.phs_add_spans(sim.h, 0, [0], [1e-3])                    # the topology has no compute lanes
    assert e.value.code == B.PHS_EINVAL
    sim.close()
    sim = B.Sim(W.topo_desc(W.TOPO_SINGLE, 2, 4, compute_lanes=1), batch=1)
    assert B.phs_num_links(sim.h) == 32 + 8
    for kw in (dict(gpu=[9], duration=[1e-3]), dict(gpu=[0], duration=[0.0]), dict(gpu=[0], duration=[1e-3], lane=[1]),
               dict(gpu=[0], duration=[1e-3], dep_off=[0, 1], dep_ids=[0])):
        with pytest.raises(B.PhsError) as e:
            B.phs_add_spans(sim.h, 0, **kw)
        assert e.value.code == B.PHS_EINVAL
    assert B.phs_add_spans(sim.h, 0, [0, 1], [1e-3, 2e-3]) == 0
    with pytest.raises(B.PhsError):
        B.phs_add_collective(sim.h, 0, B.ALLGATHER_RING, [0, 1, 2], 1e6, after_flows=[5])      # not an earlier flow
    sim.close()


def test_graph_topology_equals_the_oracle():
    """NEXT-4: user-supplied link list with shortest-path ECMP -- routes, latencies, DAG equal the oracle's."""
    _compare_tables(W.graph_fabric(batch=3))
    _compare_tables(W.graph_fabric(batch=2, n_gpus=32, gpus_per_leaf=8, n_spines=4, seed0=1))
    g = W.graph_fabric(batch=1).desc["graph"]
    for bad in (dict(n_gpus=1), dict(n_nodes=3), dict(link_to=np.where(np.arange(len(g["link_to"])) == 0, 999, g["link_to"])),
                dict(cap_Bps=np.where(np.arange(len(g["cap_Bps"])) == 3, 0.0, g["cap_Bps"]))):
        with pytest.raises(B.PhsError) as e:
            B.phs_create_topology(dict(graph=dict(g, **bad)), 0, 1)
        assert e.value.code == B.PHS_EINVAL
    # two GPUs eight switches apart: refused when the flow is added, nothing half-added
    n = 10
    lf = [0] + list(range(2, n)) + [1]; lt = list(range(2, n)) + [1] + [0]
    sim = B.Sim(W.graph_desc(2, n, lf, lt, [1e9] * len(lf), [0.0] * len(lf)), batch=1)
    with pytest.raises(B.PhsError) as e:
        B.phs_add_flows(sim.h, 0, [0], [1], [1.0])
    assert e.value.code == B.PHS_EINVAL and sim.num_flows(0) == 0
    B.phs_add_flows(sim.h, 0, [1], [0], [1e3])
    assert list(sim.paths(0)[1]) == [len(lf) - 1]
    sim.close()


def test_set_devices_is_validated_on_the_host():
    w = W.cfg3(batch=3)
    sim = B.Sim.from_workload(w)
    for bad in ([], [-1], [0, 0, 0, 0]):                # empty, negative id, more devices than instances
        with pytest.raises((B.PhsError, ValueError, TypeError)):
            B.phs_set_devices(sim.h, bad)
    B.phs_set_devices(sim.h, [0, 0])
    with pytest.raises(B.PhsError) as e:                # no CUDA device here: the shards fail loudly, nothing falls back
        sim.run()
    assert e.value.code == B.PHS_ECUDA
    sim.close()


def test_deferred_expansion_keeps_submission_order():
    """phs_add_collective records the collective and its flows are expanded later (by the next raw-flow submission,
    a table getter, or phs_finalize).  Flow ids must still follow submission order, and reading tables between
    submissions must not change what is finally built."""
    d = W.topo_desc(W.TOPO_LEAF_SPINE, 4, 4, n_leaves=2, n_spines=2, uplinks_per_leaf_spine=2)
    ring = np.array([1, 6, 11, 12, 3], np.int32)

    def submit(h, peek):
        a = B.phs_add_collective(h, 0, B.ALLREDUCE_RING, ring, 5e6, 1e-5)
        assert a == 0 and B.phs_num_flows(h, 0) == 2 * 4 * 5          # counted before it is expanded
        if peek:
            off, _links = B.phs_get_paths(h, 0)
            assert len(off) == 41
        first = B.phs_add_flows(h, 0, [0, 2], [9, 13], [1e5, 2e5], dep_off=[0, 1, 3], dep_ids=[39, 0, 38])
        assert first == 40                                            # raw flows come after the ring's 40 flows
        b = B.phs_add_collective(h, 0, B.ALLTOALL, [0, 5, 10, 15], 3e6, 0.0, after=[0])
        if peek:
            B.phs_get_preds(h, 0)
        c = B.phs_add_collective(h, 0, B.ALLGATHER_RING, [15, 5, 0], 2e6, 0.0, after=[b])
        assert (b, c) == (1, 2) and B.phs_num_flows(h, 0) == 40 + 2 + 12 + 6
        return B.phs_get_paths(h, 0), B.phs_get_preds(h, 0), B.phs_get_flow_table(h, 0)

    h1, h2 = B.phs_create_topology(d, 3, 1), B.phs_create_topology(d, 3, 1)
    t1, t2 = submit(h1, peek=True), submit(h2, peek=False)
    for x, y in zip(t1, t2):
        for u, v in zip(x, y):
            assert np.array_equal(u, v)
    # ring step s > 0 repeats the path of step 0 (ECMP keys on pair + collective)
    off, links = t1[0]
    for s_ in range(1, 8):
        for i in range(5):
            f0, f = i, s_ * 5 + i
            assert np.array_equal(links[off[f]:off[f + 1]], links[off[f0]:off[f0 + 1]])
    B.phs_destroy(h1)
    B.phs_destroy(h2)


def test_batched_capacities_equal_per_instance_calls():
    w = W.cfg3(batch=5)
    h = B.phs_create_topology(w.desc, 0, 5)
    L = B.phs_num_links(h)
    m = W.capacity_matrix(w.desc, w.instances, L)
    assert m.shape == (5, L)
    for i, inst in enumerate(w.instances):
        assert np.array_equal(m[i], inst.capacities(w.desc, L))     # the vectorised form of Instance.capacities
    B.phs_set_link_capacities_batch(h, m)
    for i in range(5):
        assert np.array_equal(B.phs_get_link_capacities(h, i), m[i])
    bad = m.copy()
    bad[3, 7] = 0.0
    with pytest.raises(B.PhsError) as e:
        B.phs_set_link_capacities_batch(h, bad)
    assert e.value.code == B.PHS_EINVAL
    assert np.array_equal(B.phs_get_link_capacities(h, 0), m[0])    # a refused call changes nothing
    with pytest.raises(ValueError):
        B.phs_set_link_capacities_batch(h, m[:4])
    B.phs_destroy(h)


def test_input_validation_and_state_errors():
    d = W.topo_desc(W.TOPO_SINGLE, 2, 8)
    h = B.phs_create_topology(d, 0, 2)
    for bad in [lambda: B.phs_add_flows(h, 0, [0], [0], [1.0]),
                lambda: B.phs_add_flows(h, 0, [0], [1], [0.0]),
                lambda: B.phs_add_flows(h, 0, [0], [1], [float("nan")]),
                lambda: B.phs_add_flows(h, 0, [0], [99], [1.0]),
                lambda: B.phs_add_flows(h, 5, [0], [1], [1.0]),
                lambda: B.phs_add_collective(h, 0, B.ALLREDUCE_RING, [0, 1, 1], 1e6),
                lambda: B.phs_add_collective(h, 0, B.ALLREDUCE_RING, [0], 1e6),
                lambda: B.phs_add_collective(h, 0, 9, [0, 1], 1e6),
                lambda: B.phs_add_collective(h, 0, B.ALLREDUCE_RING, [0, 1], 1e6, after=[0]),
                lambda: B.phs_add_flows(h, 0, [0], [1], [1.0], dep_off=[0, 1], dep_ids=[0])]:
        with pytest.raises(B.PhsError) as e:
            bad()
        assert e.value.code == B.PHS_EINVAL
    assert B.phs_num_flows(h, 0) == 0 and B.phs_num_flows(h, 1) == 0
    assert B.phs_add_collective(h, -1, B.ALLGATHER_RING, [0, 1, 2], 3e6) == 0
    assert B.phs_num_flows(h, 0) == 6 and B.phs_num_flows(h, 1) == 6
    with pytest.raises(B.PhsError) as e:
        B.phs_get_completion_times(h, 0)
    assert e.value.code == B.PHS_ESTATE
    with pytest.raises(B.PhsError):
        B.phs_create_topology(dict(d, n_hosts=0), 0, 1)
    with pytest.raises(B.PhsError):
        B.phs_create_topology(W.topo_desc(W.TOPO_FAT_TREE, 7, 2, k=4, agg_uplinks=1), 0, 1)
    B.phs_destroy(h)


def test_no_cpu_fallback_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    w = W.cfg0()
    sim = B.Sim.from_workload(w)
    with pytest.raises(B.PhsError) as e:
        sim.run()
    assert e.value.code == B.PHS_ECUDA
    sim.close()


def test_run_static_needs_a_finalized_handle():
    """phs_run_static builds nothing and allocates nothing: on a handle that is not finalized it is a state error
    (checked before any CUDA call, so this runs without a GPU), and the output size must match."""
    sim = B.Sim.from_workload(W.cfg0())
    with pytest.raises(B.PhsError) as e:
        sim.run_static()
    assert e.value.code == B.PHS_ESTATE and "phs_finalize" in str(e.value)
    with pytest.raises(B.PhsError) as e:
        B.phs_run_static(None, None, None, 0)
    assert e.value.code == B.PHS_EINVAL
    sim.close()
    assert B.PHS_STATIC_SCRATCH_BYTES == 8 << 20 and B.PHS_STATIC_MAX_UNITS == 4096
    hdr = open(os.path.join(ROOT, "include", "phs.h")).read()
    assert "#define PHS_STATIC_SCRATCH_BYTES (8u << 20)" in hdr and "#define PHS_STATIC_MAX_UNITS 4096" in hdr


def test_world_size_2_sharding_over_gloo():
    """N>1 path of bench.py: instances are sharded round-robin over ranks with no data-path collective; only the
    timing max and the counts are reduced.  Run the sharding + reduction logic on CPU over gloo."""
    import subprocess
    import sys
    env = dict(os.environ, PHS_ROOT=ROOT, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29533",
                        os.path.join(ROOT, "tests", "_gloo_shard_worker.py")],
                       env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
