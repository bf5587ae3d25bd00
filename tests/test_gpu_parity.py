"""GPU parity: the CUDA path (through the C-ABI) against the CPU oracle, element by element, on the same seeded
inputs.  Bar (BASELINE.json north_star): completion times within 1e-9 relative -- and in
fact bit-equal, because both sides do the same IEEE operations in the same order per flow and every reduction is
an integer count or a min; completion order identical (ties by flow id); bottleneck ids and the event log
(time, completions, activations, filling iterations, first bottleneck) exact."""
import os

import numpy as np
import pytest

from oracle import orc
from paper_2505_01616_b200 import binding as B
from paper_2505_01616_b200 import workloads as W
from util import completion_order, oracle_build, oracle_run

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(__file__), "golden")
CTA, CLUSTER, WINDOW, GRID = 1, 2, 3, 4


def assert_instance_matches(sim, i, o, check_log=True):
    t, to = sim.completion_times(i), o.completion_times()
    assert not np.isnan(t).any()
    np.testing.assert_allclose(t, to, rtol=1e-9, atol=0)           # the stated bar
    assert np.array_equal(t, to), "completion times are expected to be bit-equal"
    assert np.array_equal(completion_order(t), completion_order(to))
    assert np.array_equal(sim.bottlenecks(i), o.bottlenecks())
    assert np.array_equal(sim.collective_times(i), o.collective_times()) or o.num_collectives == 0
    if check_log:
        ev, evo = sim.event_log(i), o.event_log()
        assert len(ev) == len(evo)
        for k in ("t", "n_completed", "n_activated", "n_rounds", "first_bneck"):
            assert np.array_equal(ev[k], evo[k]), k


def run_and_compare(w, path=0, cta_slots=0, first=0, count=None, mode=orc.MODE_FAST, expect_path=None):
    count = w.batch if count is None else count
    sim = B.Sim.from_workload(w, event_log=True, instances=(first, count), path=path, cta_slots=cta_slots)
    sim.run()
    for i in range(count):
        o = oracle_run(w.desc, w.instances[first + i], mode=mode, base_seed=w.base_seed)
        assert_instance_matches(sim, i, o)
        if expect_path:
            assert sim.path_of(i) == expect_path
    c = sim.counters()
    assert c["n_flow_events"] == 2 * sim.total_flows
    sim.close()
    # the same without the event log: the production configuration, in which an instance is decomposed into
    # independent units (reading R-LZ makes that bit-identical) and unchanged components are not re-solved
    for decompose in (True, False):
        sim = B.Sim.from_workload(w, instances=(first, count), path=path, cta_slots=cta_slots, decompose=decompose)
        sim.run()
        for i in range(count):
            o = oracle_run(w.desc, w.instances[first + i], mode=mode, base_seed=w.base_seed)
            assert_instance_matches(sim, i, o, check_log=False)
        sim.close()
    return c


@pytest.mark.parametrize("path", [CTA, CLUSTER])
def test_cfg0_full(path):
    run_and_compare(W.cfg0(), path=path, mode=orc.MODE_NAIVE, expect_path="cta" if path == CTA else "cluster")


def test_cfg1_instances_cta():
    # instance 0 (16 MiB / 1 GiB, symmetric: exact ties everywhere) and three log-uniform ones; 5632 flows each
    run_and_compare(W.cfg1(batch=4), path=0, expect_path="cta")


def _full_batch_sampled(w, sample):
    """The whole batch in the launch configuration bench.py times (no log, decomposed); sampled instances against
    the oracle element by element, every instance's flow-event count through the counters."""
    sim = B.Sim.from_workload(w)
    sim.run()
    for i in sample:
        o = oracle_run(w.desc, w.instances[i], mode=orc.MODE_FAST, base_seed=w.base_seed)
        assert_instance_matches(sim, i, o, check_log=False)
        assert sim.path_of(i) == "cta"
    c = sim.counters()
    assert c["n_flow_events"] == 2 * sim.total_flows
    t = B.phs_get_all_completion_times(sim.h)
    assert np.isfinite(t).all() and (t > 0).all()
    sim.close()


def test_cfg1_full_batch_as_benchmarked():
    _full_batch_sampled(W.cfg1(), [0, 1, 17, 42, 63])


def test_cfg3_full_batch_as_benchmarked():
    # 4,096 instances = 36,864 units: the scheduler's many-units configuration (64 threads per CTA)
    _full_batch_sampled(W.cfg3(), [0, 1, 777, 2048, 3333, 4095])


def test_cfg1_instance_cluster():
    run_and_compare(W.cfg1(batch=2), path=CLUSTER, first=1, count=1, expect_path="cluster")


def test_cfg3_instances_cta():
    run_and_compare(W.cfg3(batch=6), path=0, expect_path="cta")


def test_cfg3_seed_is_instance_index_in_sub_batches():
    run_and_compare(W.cfg3(batch=40), first=37, count=3)


@pytest.mark.parametrize("path", [CTA, CLUSTER])
def test_cfg2_shrunken_fat_tree(path):
    # k=8: 128 GPUs, 3-tier paths of 2/4/6 hops, staggered start times, AR + AG + RS mix; ragged tails everywhere
    run_and_compare(W.cfg2(k=8, agg_uplinks=2), path=path)


@pytest.mark.parametrize("path", [CTA, CLUSTER])
def test_cfg4_shrunken_alltoall(path):
    # 64 GPUs, 4032 concurrent Zipf flows, many filling rounds per event
    run_and_compare(W.cfg4(batch=2, n_hosts=8, gph=8, n_leaves=4, n_spines=2), path=path)


def _window_compare(w, gang, expect_gang=None, first=0, count=None):
    """The window path (forced: phs_set_scheduler path 3, smallest gang `gang`) against the oracle, decomposed and
    not, plus against the library's own one-event-per-iteration schedule."""
    count = w.batch if count is None else count
    for decompose in (True, False):
        sim = B.Sim.from_workload(w, instances=(first, count), path=WINDOW, cta_slots=gang, decompose=decompose)
        sim.run()
        c = sim.counters()
        assert c["window_gang"] >= 1
        if expect_gang and not decompose:      # the smallest gang asked for, or a larger one if that does not fit
            assert c["window_gang"] >= expect_gang, c
        assert c["n_windows"] <= c["n_events"] or c["window_gang"] > 1
        for i in range(count):
            o = oracle_run(w.desc, w.instances[first + i], mode=orc.MODE_FAST, base_seed=w.base_seed)
            assert_instance_matches(sim, i, o, check_log=False)
        if not decompose:
            assert all(sim.path_of(i) == "window" for i in range(count))
        sim.close()


@pytest.mark.parametrize("gang", [1, 4])
def test_window_path_ring_configs(gang):
    # cfg1 (TP + DP rings that contend on the leaf-spine uplinks), cfg3 (random capacities, chained collectives)
    _window_compare(W.cfg1(batch=3, n_hosts=8, gph=4, n_leaves=4, n_spines=2), gang, expect_gang=gang)
    _window_compare(W.cfg3(batch=4), gang, expect_gang=gang)
    _window_compare(W.cfg1(batch=2), gang, first=1, count=1, expect_gang=gang)


@pytest.mark.parametrize("gang", [1, 2, 8, 16])
def test_window_path_shrunken_fat_tree(gang):
    # k=8 fat tree, staggered starts, AR + AG + RS: many events per window (the regime the path is built for)
    _window_compare(W.cfg2(k=8, agg_uplinks=2), gang, expect_gang=gang)


def test_window_path_single_component_and_raw_flows():
    # all-to-all: ONE component, no dependencies (lmin = +inf: a single window); a gang has nothing to share out
    _window_compare(W.cfg4(batch=2, n_hosts=4, gph=4, n_leaves=2, n_spines=2), 4, expect_gang=1)
    _window_compare(W.cfg0(), 1, expect_gang=1)
    # too large for the shared memory of one CTA, and one component cannot be shared out: not on the window path
    w = W.cfg4(batch=1, n_hosts=8, gph=8, n_leaves=4, n_spines=2)
    sim = B.Sim.from_workload(w, path=WINDOW, cta_slots=4, decompose=False)
    sim.run()
    assert sim.path_of(0) != "window"
    assert_instance_matches(sim, 0, oracle_run(w.desc, w.instances[0], mode=orc.MODE_FAST), check_log=False)
    sim.close()


def test_window_path_is_chosen_for_dense_units_only():
    # automatic policy: shrunken cfg2 (events every few hundred ns against a 4 us lookahead) goes to the window path,
    # cfg1 / cfg3 (events tens of us apart) stay one event per iteration
    sim = B.Sim.from_workload(W.cfg2(k=8, agg_uplinks=2))
    sim.run()
    assert sim.path_of(0) == "window" and sim.counters()["n_windows"] < sim.counters()["n_events"]
    sim.close()
    sim = B.Sim.from_workload(W.cfg3(batch=2))
    sim.run()
    assert sim.path_of(0) == "cta" and sim.counters()["window_gang"] == 0
    sim.close()
    # the window schedule switched off: same results, CTA / cluster paths only
    a = B.Sim.from_workload(W.cfg2(k=8, agg_uplinks=2), windows=False)
    a.run()
    assert a.path_of(0) != "window"
    o = oracle_run(W.cfg2(k=8, agg_uplinks=2).desc, W.cfg2(k=8, agg_uplinks=2).instances[0], mode=orc.MODE_FAST)
    assert_instance_matches(a, 0, o, check_log=False)
    a.close()


def test_chain_and_tree_collectives_on_every_path():
    """NEXT-3: pipelined chain broadcast / reduce and binary-tree all-reduce, mixed with ring
    collectives through `after` edges, on a leaf-spine fabric (contention on the uplinks), on all four kernel paths."""
    d = W.topo_desc(W.TOPO_LEAF_SPINE, 8, 4, fabric_Bps=W.gbps(400.0), n_leaves=4, n_spines=2, uplinks_per_leaf_spine=1)
    rng = np.random.default_rng(77)
    insts = []
    for i in range(3):
        perm = rng.permutation(32).astype(np.int32)
        ops = [W.Coll(W.BROADCAST_CHAIN, perm[:9], 8e6, 0.0, (), 5),
               W.Coll(W.ALLREDUCE_TREE, perm[4:17], 6e6, 1e-5, (), 3),
               W.Coll(W.REDUCE_CHAIN, perm[10:20], 4e6, 0.0, (0,), 4),
               W.Coll(W.ALLREDUCE_RING, perm[:8], 16e6, 0.0, (1, 2)),
               W.Coll(W.ALLREDUCE_TREE, perm[2:9], 2e6, 0.0, (3,), 1),
               W.Coll(W.ALLTOALL, perm[20:28], 3e6, 2e-5, (1,)),
               W.Coll(W.BROADCAST_CHAIN, perm[18:30], 5e6, 0.0, (5, 4), 2)]
        insts.append(W.Instance(seed=i, ops=ops))
    w = W.Workload("next3", d, 11, insts)
    for path in (0, CTA, CLUSTER):
        run_and_compare(w, path=path)
    _window_compare(w, 2)
    _grid_compare(w)


def test_compute_spans_training_step_on_every_path():
    """NEXT-2 (PAPER.md L84 / L206): compute spans in the DAG, overlapping the collectives; zero-latency engine links, so
    released spans activate within the releasing event."""
    w = W.train_step(batch=3, n_hosts=4, gph=4, layers=3, buckets=2)
    for path in (0, CTA, CLUSTER):
        run_and_compare(w, path=path)
    _grid_compare(w)
    # a span alone ends at exactly start + duration on the GPU as well
    sim = B.Sim(W.topo_desc(W.TOPO_SINGLE, 1, 8, compute_lanes=2), batch=1)
    B.phs_add_spans(sim.h, 0, [0, 5, 5], [1e-3, 3.3e-4, 7e-5], lane=[0, 0, 1], start=[0.0, 1e-4, 2.5e-4])
    sim.run()
    assert list(sim.completion_times(0)) == [1e-3, 1e-4 + 3.3e-4, 2.5e-4 + 7e-5]
    sim.close()


def test_graph_topology_on_every_path():
    """NEXT-4: a user-supplied topology with per-link capacities and latencies."""
    w = W.graph_fabric(batch=3)
    for path in (0, CTA, CLUSTER):
        run_and_compare(w, path=path)
    _grid_compare(w)


def test_cta_slot_overflow_falls_back_to_cluster():
    w = W.cfg4(batch=3, n_hosts=4, gph=8, n_leaves=2, n_spines=2)      # 992 flows pending at t=0 > 64 slots
    sim = B.Sim.from_workload(w, event_log=True, cta_slots=64)
    sim.run()
    for i in range(3):
        assert sim.path_of(i) == "cluster"
        assert_instance_matches(sim, i, oracle_run(w.desc, w.instances[i], mode=orc.MODE_FAST))
    sim.run()                                                           # second run goes straight to the cluster path
    assert_instance_matches(sim, 1, oracle_run(w.desc, w.instances[1], mode=orc.MODE_FAST))
    sim.close()


def test_rerun_is_idempotent_and_batch_position_independent():
    w = W.cfg3(batch=5)
    a = B.Sim.from_workload(w)
    a.run()
    t1 = [a.completion_times(i) for i in range(5)]
    a.run()
    for i in range(5):
        assert np.array_equal(a.completion_times(i), t1[i])
    b = B.Sim.from_workload(w, instances=(3, 2))
    b.run()
    assert np.array_equal(b.completion_times(0), t1[3]) and np.array_equal(b.completion_times(1), t1[4])
    a.close(); b.close()


def test_edge_cases():
    d = W.topo_desc(W.TOPO_SINGLE, 2, 8)
    # empty instance next to a non-empty one; zero-latency chain; a flow that can never start (cycle-free API, so
    # "never" = waits on nothing -> fine); simultaneous bit-equal completions
    sim = B.Sim(d, batch=3, event_log=True)
    B.phs_add_flows(sim.h, 1, [0, 1, 2], [8, 8, 8], [1e6, 2e6, 4e6])
    B.phs_add_collective(sim.h, 2, B.ALLTOALL, np.arange(16, dtype=np.int32), 1e6)
    sim.run()
    assert sim.num_flows(0) == 0 and len(sim.completion_times(0)) == 0 and len(sim.event_log(0)) == 0
    o = orc.Sim(d, 1); o.add_flows([0, 1, 2], [8, 8, 8], [1e6, 2e6, 4e6]); o.run()
    assert_instance_matches(sim, 1, o)
    o = orc.Sim(d, 2); o.add_collective(orc.ALLTOALL, np.arange(16, dtype=np.int32), 1e6); o.run()
    assert_instance_matches(sim, 2, o)
    sim.close()
    d0 = W.topo_desc(W.TOPO_SINGLE, 2, 8, hop_latency_s=0.0)
    sim = B.Sim(d0, batch=1, event_log=True)
    n = 50
    src = np.arange(n) % 16
    dst = (src + 3) % 16
    dep_off = np.concatenate([[0], np.arange(n)])          # flow i waits for flow i-1: a zero-latency chain
    dep_ids = np.arange(n - 1)
    B.phs_add_flows(sim.h, 0, src, dst, np.full(n, 1e5), None, dep_off, dep_ids)
    sim.run()
    o = orc.Sim(d0, 0); o.add_flows(src, dst, np.full(n, 1e5), None, dep_off, dep_ids); o.run()
    assert_instance_matches(sim, 0, o)
    sim.close()


def test_device_output_pointer():
    import torch
    w = W.cfg0()
    sim = B.Sim.from_workload(w)
    st = torch.cuda.Stream()
    sim.run(stream=st.cuda_stream)
    out = torch.empty(sim.num_flows(0), dtype=torch.float64, device="cuda")
    B.phs_get_completion_times(sim.h, 0, device_ptr=out.data_ptr())
    st.synchronize()
    assert np.array_equal(out.cpu().numpy(), sim.completion_times(0))
    sim.close()


def _golden(name):
    z = np.load(os.path.join(GOLD, name))
    return z


def _check_against_golden(sim, inst, z):
    import hashlib
    t, b = sim.completion_times(inst), sim.bottlenecks(inst)
    assert np.array_equal(t[z["idx"]], z["t_done"])
    assert np.array_equal(b[z["idx"]], z["bneck"])
    assert hashlib.sha256(t.tobytes()).hexdigest() == z["sha_t"].item()
    assert hashlib.sha256(b.tobytes()).hexdigest() == z["sha_bneck"].item()


def _check_log_against_golden(sim, inst, z):
    import hashlib
    ev = sim.event_log(inst)
    assert len(ev) == int(z["n_events"])
    assert hashlib.sha256(np.ascontiguousarray(ev["t"]).tobytes()).hexdigest() == z["sha_event_t"].item()


def test_cfg4_full_size_whole_batch_as_benchmarked():
    """BASELINE.json configs[4] at full size, all 8 instances in the launch bench.py times (W.cfg4(), no log,
    scheduler on automatic), every instance against the stored oracle output (4096 sampled flows, SHA-256 of all
    completion times and of all bottleneck ids).  The expected values were written by tests/golden/make_golden.py,
    which calls only oracle/ (fast mode).  Then the same batch with the event log on: event count and SHA-256 of the
    log's time column per instance."""
    w = W.cfg4()
    assert w.batch == 8
    zs = [_golden(f"cfg4_inst{i}.npz") for i in range(w.batch)]
    sim = B.Sim.from_workload(w)
    sim.run()
    for i in range(w.batch):
        _check_against_golden(sim, i, zs[i])
    c = sim.counters()
    assert c["n_flow_events"] == 2 * sim.total_flows
    if c["cluster_size"] > 0 and sim.path_of(0) == "cluster":
        # more units than resident clusters: some cluster simulated two units back to back (ticket, re-init, scratch reuse)
        print("cfg4 launch: cluster size", c["cluster_size"], "resident", c["clusters_resident"])
    sim.close()
    sim = B.Sim.from_workload(w, event_log=True)
    sim.run()
    for i in range(w.batch):
        _check_against_golden(sim, i, zs[i])
        _check_log_against_golden(sim, i, zs[i])
    sim.close()


def test_cfg2_full_size_as_benchmarked():
    """BASELINE.json configs[2] at full size (1,069,056 flows in one instance) in the launch configuration bench.py
    uses, against the stored oracle output."""
    z = _golden("cfg2_inst0.npz")
    w = W.cfg2()
    sim = B.Sim.from_workload(w)
    sim.run()
    _check_against_golden(sim, 0, z)
    c = sim.counters()
    assert c["n_flow_events"] == 2 * sim.total_flows
    # the 1.04 M-flow data-parallel unit runs the lookahead-window schedule: far fewer loop iterations than events
    assert sim.path_of(0) == "window" and c["n_events"] < int(z["n_events"]) // 10
    sim.close()


def _grid_compare(w, first=0, count=None, decompose=False):
    """The grid path (forced: phs_set_scheduler path 4; it does not write the event log) against the oracle."""
    count = w.batch if count is None else count
    sim = B.Sim.from_workload(w, instances=(first, count), path=GRID, decompose=decompose)
    sim.run()
    c = sim.counters()
    assert c["grid_ctas"] >= 1
    for i in range(count):
        o = oracle_run(w.desc, w.instances[first + i], mode=orc.MODE_FAST, base_seed=w.base_seed)
        assert_instance_matches(sim, i, o, check_log=False)
        assert sim.path_of(i) == "grid"
    sim.close()


def test_grid_path_small_configs():
    _grid_compare(W.cfg0())
    _grid_compare(W.cfg1(batch=2, n_hosts=8, gph=4, n_leaves=4, n_spines=2))
    _grid_compare(W.cfg3(batch=2), decompose=True)            # several units, one after the other
    _grid_compare(W.cfg2(k=4, agg_uplinks=1))
    _grid_compare(W.cfg4(batch=1, n_hosts=8, gph=8, n_leaves=4, n_spines=2))      # many rounds per event


def test_unit_larger_than_a_cluster_runs_on_the_whole_grid():
    """BASELINE.json north_star: "the whole grid to each large instance".  A unit whose concurrent flows exceed the
    shared memory of 16 SMs used to be refused (PHS_ERANGE); the scheduler now hands it to the grid path.  Uniform
    304-GPU all-to-all (92,112 concurrent flows, P8: every flow B/(N-1)) against the oracle run live."""
    d = W.topo_desc(W.TOPO_SINGLE, 38, 8)                      # 304 GPUs on one switch
    ranks = np.arange(304, dtype=np.int32)
    sim = B.Sim(d, batch=1)
    B.phs_add_collective(sim.h, 0, B.ALLTOALL, ranks, 304e6)
    sim.run()
    assert sim.path_of(0) == "grid" and sim.counters()["grid_ctas"] > 100
    o = orc.Sim(d, 0)
    o.add_collective(orc.ALLTOALL, ranks, 304e6)
    o.run(mode=orc.MODE_FAST)
    assert_instance_matches(sim, 0, o, check_log=False)
    sim.run()                                                   # later runs go straight to the grid path
    assert_instance_matches(sim, 0, o, check_log=False)
    sim.close()
    with_log = B.Sim(d, batch=1, event_log=True)                # the grid path does not write the event log
    B.phs_add_collective(with_log.h, 0, B.ALLTOALL, ranks, 304e6)
    with pytest.raises(B.PhsError) as e:
        with_log.run()
    assert e.value.code == B.PHS_ERANGE
    with_log.close()


def test_grid_path_skewed_alltoall_92k_flows_against_stored_oracle():
    """cfg4's recipe on 304 GPUs: 92,112 concurrent Zipf-skewed flows, ~92 K events with many filling rounds each --
    fits no cluster.  Expected values written by tests/golden/make_golden.py a2a304 (oracle only)."""
    path = os.path.join(GOLD, "a2a304_inst0.npz")
    if not os.path.exists(path):
        pytest.skip("golden file not generated")
    w = W.cfg4(batch=1, n_hosts=38, gph=8, n_leaves=2, n_spines=4)
    sim = B.Sim.from_workload(w, decompose=False)
    sim.run()
    assert sim.path_of(0) == "grid"
    _check_against_golden(sim, 0, _golden("a2a304_inst0.npz"))
    sim.close()


def test_decomposition_knob_state_and_counters():
    w = W.cfg1(batch=2, n_hosts=8, gph=4, n_leaves=4, n_spines=2)
    a = B.Sim.from_workload(w)                       # decomposed: TP rings and the DP group are separate units
    b = B.Sim.from_workload(w, decompose=False)
    a.run(); b.run()
    for i in range(2):
        assert np.array_equal(a.completion_times(i), b.completion_times(i))
        assert np.array_equal(a.bottlenecks(i), b.bottlenecks(i))
        assert np.array_equal(a.collective_times(i), b.collective_times(i))
    assert a.counters()["n_events"] >= b.counters()["n_events"]      # coinciding events count once per unit
    with pytest.raises(B.PhsError) as e:
        B.phs_set_decomposition(a.h, False)
    assert e.value.code == B.PHS_ESTATE
    a.close(); b.close()


@pytest.mark.parametrize("seed", range(6))
def test_random_dags_of_raw_flows(seed):
    """Differential test on irregular inputs: raw flows with random dependencies (fan-in up to 24, fan-out beyond the
    two inline successors), random start times, a mix of zero and non-zero latency, groups that decompose into many
    small units, on both kernel paths, with and without the event log."""
    rng = np.random.default_rng(1000 + seed)
    lat = [0.0, 1e-6][seed % 2]
    if seed % 3 == 0:
        d = W.topo_desc(W.TOPO_SINGLE, 4, 8, hop_latency_s=lat)
    elif seed % 3 == 1:
        d = W.topo_desc(W.TOPO_LEAF_SPINE, 8, 4, hop_latency_s=lat, fabric_Bps=W.gbps(400.0), n_leaves=4, n_spines=2,
                        uplinks_per_leaf_spine=1)
    else:
        d = W.topo_desc(W.TOPO_FAT_TREE, 8, 2, hop_latency_s=lat, fabric_Bps=W.gbps(400.0), k=4, agg_uplinks=1)
    G = d["n_hosts"] * d["gpus_per_host"]
    insts = []
    for i in range(3):
        n = int(rng.integers(200, 900))
        src = rng.integers(0, G, n).astype(np.int32)
        dst = ((src + rng.integers(1, G, n)) % G).astype(np.int32)
        if i == 2:                                   # many small independent groups: traffic stays inside GPU pairs
            src = (2 * rng.integers(0, G // 2, n)).astype(np.int32)
            dst = (src + 1).astype(np.int32)
        nbytes = np.floor(np.exp(rng.uniform(np.log(1e3), np.log(5e7), n)))
        start = np.where(rng.random(n) < 0.3, rng.uniform(0, 2e-3, n), 0.0)
        dep_off, dep_ids = [0], []
        for f in range(n):
            k = 0 if f == 0 else int(rng.choice([0, 0, 1, 2, 3, 24], p=[0.3, 0.2, 0.25, 0.15, 0.08, 0.02]))
            lo = max(0, f - 60)
            deps = np.unique(rng.integers(lo, f, min(k, f - lo))) if k and f > lo else []
            if i == 2 and len(deps):                 # keep the small groups independent: depend within the pair
                deps = [p for p in deps if src[p] == src[f]]
            dep_ids.extend(int(x) for x in deps)
            dep_off.append(len(dep_ids))
        insts.append(W.Instance(seed=i, ops=[W.RawFlows(src, dst, nbytes, start, np.array(dep_off, np.int64),
                                                        np.array(dep_ids, np.int64))]))
    w = W.Workload("fuzz", d, 7 * seed, insts)
    run_and_compare(w, path=[0, CTA, CLUSTER][seed % 3], mode=orc.MODE_FAST)
    if lat > 0.0:       # the window path needs a positive lookahead; fan-in up to 24 exercises the release lists
        _window_compare(w, [1, 2, 4][seed % 3])


@pytest.mark.parametrize("path", [CTA, CLUSTER])
def test_throughput_history_equals_the_oracle(path):
    """NEXT-1 groundwork (PAPER.md L128 / L167): the per-flow list of (time, new rate) rate changes.  Bit-equal to the
    oracle's, with and without decomposition, and it reconstructs every flow's bytes."""
    w = W.cfg1(batch=2, n_hosts=8, gph=4, n_leaves=4, n_spines=2)
    for decompose in (True, False):
        sim = B.Sim.from_workload(w, path=path, decompose=decompose, history=1 << 20)
        sim.run()
        for i in range(w.batch):
            o = oracle_run(w.desc, w.instances[i], mode=orc.MODE_FAST)
            fl, t, r = o.history()
            off, tg, rg = sim.history(i)
            assert off[-1] == len(fl)
            assert np.array_equal(np.diff(off), np.bincount(fl, minlength=o.num_flows))
            assert np.array_equal(tg, t) and np.array_equal(rg, r)
            td, nbytes = sim.completion_times(i), o.flows()[2]
            for f in range(0, o.num_flows, 37):      # constant-throughput intervals add up to the flow's size
                tt = np.append(tg[off[f]:off[f + 1]], td[f])
                assert abs(np.sum(rg[off[f]:off[f + 1]] * np.diff(tt)) - nbytes[f]) <= 1e-9 * nbytes[f]
        sim.close()
    small = B.Sim.from_workload(w, path=path, history=100)           # too small: refused, with the count needed
    with pytest.raises(B.PhsError) as e:
        small.run()
    assert e.value.code == B.PHS_ERANGE and "needs" in str(e.value)
    small.close()


@pytest.mark.parametrize("path", [CTA, CLUSTER])
def test_run_until_stops_where_the_oracle_stops(path):
    """PAPER.md L167 "advancing the simulation ... up to a specified time": completion times, bottlenecks, collective
    times (NaN / -1 for what has not finished), event log and throughput history up to t_stop, bit-equal to the oracle
    stopped at the same time."""
    w = W.cfg1(batch=2, n_hosts=8, gph=4, n_leaves=4, n_spines=2)
    full = [oracle_run(w.desc, w.instances[i], mode=orc.MODE_FAST).completion_times() for i in range(w.batch)]
    t_end = max(t.max() for t in full)
    for frac in (0.0, 0.31, 0.77, 2.0):
        t_stop = frac * t_end
        for log, decompose in ((True, False), (False, True)):
            sim = B.Sim.from_workload(w, path=path, event_log=log, decompose=decompose, history=1 << 20)
            sim.run(until=t_stop)
            for i in range(w.batch):
                inst = w.instances[i]
                o = oracle_build(w.desc, inst)
                o.run(mode=orc.MODE_FAST, until=t_stop)
                t, to = sim.completion_times(i), o.completion_times()
                assert np.array_equal(t, to, equal_nan=True)
                assert np.isnan(to).any() == (frac < 1.0) and (frac == 0.0 or not np.isnan(to).all())
                assert np.array_equal(sim.bottlenecks(i), o.bottlenecks())
                assert np.array_equal(sim.collective_times(i), o.collective_times(), equal_nan=True)
                fl, th, rh = o.history()
                off, tg, rg = sim.history(i)
                assert np.array_equal(np.diff(off), np.bincount(fl, minlength=o.num_flows))
                assert np.array_equal(tg, th) and np.array_equal(rg, rh)
                if log:
                    assert np.array_equal(sim.event_log(i), o.event_log())
            sim.close()


@pytest.mark.parametrize("path", [0, CLUSTER])
def test_run_until_resumes_from_the_parked_state(path):
    """Successive phs_run_until calls with growing stop times continue the units from where they stopped (shared
    memory and registers parked in global memory, on both kernel paths); the result at every stop equals the oracle
    stopped there, and the final state equals a single full run."""
    w = W.cfg3(batch=3)
    ref = [oracle_run(w.desc, w.instances[i], mode=orc.MODE_FAST) for i in range(w.batch)]
    t_end = max(o.completion_times().max() for o in ref)
    for log, decompose in ((False, True), (True, False)):
        sim = B.Sim.from_workload(w, event_log=log, decompose=decompose, history=1 << 21, path=path)
        prev = None
        for frac in (0.1, 0.1, 0.45, 0.8, 0.3, 1.5):           # growing, repeated, backwards, past the end
            sim.run(until=frac * t_end)
            resumed = sim.counters()["resumed_units"]
            assert (resumed > 0) == (prev is not None and frac >= prev), (frac, prev, resumed)
            prev = frac
            for i in range(w.batch):
                o = oracle_build(w.desc, w.instances[i])
                o.run(mode=orc.MODE_FAST, until=frac * t_end)
                assert np.array_equal(sim.completion_times(i), o.completion_times(), equal_nan=True), (frac, i)
                assert np.array_equal(sim.bottlenecks(i), o.bottlenecks())
                assert np.array_equal(sim.collective_times(i), o.collective_times(), equal_nan=True)
                fl, th, rh = o.history()
                off, tg, rg = sim.history(i)
                assert np.array_equal(np.diff(off), np.bincount(fl, minlength=o.num_flows))
                assert np.array_equal(tg, th) and np.array_equal(rg, rh)
                if log:
                    assert np.array_equal(sim.event_log(i), o.event_log())
        for i in range(w.batch):
            assert np.array_equal(sim.completion_times(i), ref[i].completion_times())
        sim.close()


@pytest.mark.parametrize("lean", ["1", "3"])
def test_cta_path_lean_layout(monkeypatch, lean):
    """CtaLaunch::lean (csrc/phs_device.h): in the throughput regime the scheduler moves the per-link arrays that only
    multi-round solves touch (and the capacities) from shared memory to a per-CTA global scratch, so that more CTAs
    are resident.  Forced here (PHS_CTA_LEAN) on small batches: ring traffic with single-round solves, all-to-all
    traffic with many rounds per event, several units per CTA in a row (the scratch is reused), and a run that is
    stopped and resumed (a parked unit continues on another CTA's scratch region)."""
    monkeypatch.setenv("PHS_CTA_LEAN", lean)
    for w in (W.cfg3(batch=5), W.cfg1(batch=2, n_hosts=8, gph=4, n_leaves=4, n_spines=2),
              W.cfg4(batch=3, n_hosts=8, gph=8, n_leaves=4, n_spines=2), W.cfg2(k=4, agg_uplinks=1)):
        for decompose in (True, False):
            sim = B.Sim.from_workload(w, path=CTA, decompose=decompose)
            sim.run()
            for i in range(w.batch):
                o = oracle_run(w.desc, w.instances[i], mode=orc.MODE_FAST, base_seed=w.base_seed)
                assert_instance_matches(sim, i, o, check_log=False)
            assert sim.path_of(0) in ("cta", "cluster")         # a unit that runs out of slots moves to a cluster
            sim.close()
    w = W.cfg4(batch=2, n_hosts=4, gph=8, n_leaves=2, n_spines=2)
    ref = [oracle_run(w.desc, w.instances[i], mode=orc.MODE_FAST) for i in range(w.batch)]
    t_end = max(o.completion_times().max() for o in ref)
    sim = B.Sim.from_workload(w, path=CTA, decompose=False)
    for k, frac in enumerate((0.2, 0.6, 1.2)):
        sim.run(until=frac * t_end)
        assert (sim.counters()["resumed_units"] > 0) == (k > 0)
        for i in range(w.batch):
            o = oracle_build(w.desc, w.instances[i])
            o.run(mode=orc.MODE_FAST, until=frac * t_end)
            assert np.array_equal(sim.completion_times(i), o.completion_times(), equal_nan=True), (frac, i)
            assert np.array_equal(sim.bottlenecks(i), o.bottlenecks())
    sim.close()
    sim = B.Sim.from_workload(W.cfg3(batch=5), path=CTA)
    sim.run()
    assert all(sim.path_of(i) == "cta" for i in range(5))
    sim.close()


@pytest.mark.parametrize("inc", ["1", "0"])
def test_incremental_resolve_with_flows_added_and_removed(monkeypatch, inc):
    """The incremental re-solve of the cluster and grid paths where it has to be careful: uniform
    all-to-alls (every flow of a step has the same rate: ties, many flows completing at one time), a second all-to-all
    chained behind the first (flows are ADDED to a component that is being re-solved: the limit drops to 0) and raw
    flows of random sizes that start in the middle of it -- against the oracle, and the same with the incremental
    re-solve switched off."""
    monkeypatch.setenv("PHS_CLUSTER_INC", inc)
    monkeypatch.setenv("PHS_GRID_INC", inc)
    d = W.topo_desc(W.TOPO_LEAF_SPINE, 8, 8, fabric_Bps=W.gbps(400.0), n_leaves=4, n_spines=2, uplinks_per_leaf_spine=2)
    insts = []
    for i in range(2):
        rng = np.random.default_rng(70 + i)
        n = 1500
        src = rng.integers(0, 64, n).astype(np.int32)
        dst = ((src + rng.integers(1, 64, n)) % 64).astype(np.int32)
        ops = [W.Coll(W.ALLTOALL, np.arange(64, dtype=np.int32), 64 * 3e5),
               W.Coll(W.ALLTOALL, np.arange(0, 64, 2, dtype=np.int32), 32 * 5e5, 0.0, (0,)),
               W.RawFlows(src, dst, np.floor(rng.uniform(1e4, 2e6, n)), start=rng.uniform(0.0, 4e-4, n))]
        insts.append(W.Instance(seed=i, ops=ops))
    w = W.Workload("a2a_chain", d, 3, insts)
    for path in (CLUSTER, GRID):
        sim = B.Sim.from_workload(w, path=path, decompose=False)
        sim.run()
        for i in range(w.batch):
            o = oracle_run(w.desc, w.instances[i], mode=orc.MODE_FAST, base_seed=w.base_seed)
            assert_instance_matches(sim, i, o, check_log=False)
        assert sim.path_of(0) == ("cluster" if path == CLUSTER else "grid")
        sim.close()
    # the CTA path: a batch of small instances of the same kind (the scheduler turns the incremental re-solve on when
    # most flows of the launch are all-to-all / raw flows), stopped and resumed on the way
    monkeypatch.setenv("PHS_CTA_INC", inc)
    d = W.topo_desc(W.TOPO_LEAF_SPINE, 4, 8, fabric_Bps=W.gbps(200.0), n_leaves=2, n_spines=2, uplinks_per_leaf_spine=1)
    insts = []
    for i in range(6):
        rng = np.random.default_rng(90 + i)
        n = 300
        src = rng.integers(0, 32, n).astype(np.int32)
        dst = ((src + rng.integers(1, 32, n)) % 32).astype(np.int32)
        ops = [W.Coll(W.ALLTOALL, np.arange(32, dtype=np.int32), 32 * 2e5),
               W.Coll(W.ALLTOALL, np.arange(0, 32, 2, dtype=np.int32), 16 * 4e5, 0.0, (0,)),
               W.RawFlows(src, dst, np.floor(rng.uniform(1e4, 1e6, n)), start=rng.uniform(0.0, 2e-4, n))]
        insts.append(W.Instance(seed=i, ops=ops))
    w = W.Workload("a2a_chain_small", d, 5, insts)
    ref = [oracle_run(w.desc, w.instances[i], mode=orc.MODE_FAST, base_seed=w.base_seed) for i in range(w.batch)]
    t_end = max(o.completion_times().max() for o in ref)
    sim = B.Sim.from_workload(w, path=CTA, decompose=False)
    for frac in (0.3, 0.7, 1.5):
        sim.run(until=frac * t_end)
        for i in range(w.batch):
            o = oracle_build(w.desc, w.instances[i], base_seed=w.base_seed)
            o.run(mode=orc.MODE_FAST, until=frac * t_end)
            assert np.array_equal(sim.completion_times(i), o.completion_times(), equal_nan=True), (frac, i)
            assert np.array_equal(sim.bottlenecks(i), o.bottlenecks())
    for i in range(w.batch):
        assert_instance_matches(sim, i, ref[i], check_log=False)
        assert sim.path_of(i) == "cta"
    sim.close()


def test_run_until_resumes_a_multi_cta_cluster():
    """Parking on the cluster path with several CTAs per unit (replicated shares, debit pre-aggregation): 4032
    concurrent flows per instance, stopped twice on the way."""
    w = W.cfg4(batch=2, n_hosts=8, gph=8, n_leaves=4, n_spines=2)
    sim = B.Sim.from_workload(w, path=CLUSTER, history=1 << 22)
    ref = [oracle_run(w.desc, w.instances[i], mode=orc.MODE_FAST) for i in range(w.batch)]
    t_end = max(o.completion_times().max() for o in ref)
    for k, frac in enumerate((0.2, 0.6, 1.2)):
        sim.run(until=frac * t_end)
        c = sim.counters()
        assert c["cluster_size"] > 1 and (c["resumed_units"] > 0) == (k > 0)
        for i in range(w.batch):
            o = oracle_build(w.desc, w.instances[i])
            o.run(mode=orc.MODE_FAST, until=frac * t_end)
            assert np.array_equal(sim.completion_times(i), o.completion_times(), equal_nan=True), (frac, i)
            assert np.array_equal(sim.bottlenecks(i), o.bottlenecks())
            fl, th, rh = o.history()
            off, tg, rg = sim.history(i)
            assert np.array_equal(np.diff(off), np.bincount(fl, minlength=o.num_flows))
            assert np.array_equal(tg, th) and np.array_equal(rg, rh)
    sim.close()


@pytest.mark.parametrize("path", [0, CLUSTER])
def test_time_rollback_equals_a_fresh_run(path):
    """NEXT-1 (Fig. 4; L167): the simulation has run ahead in steps (every stop keeps a snapshot of
    the parked on-chip state); then a flow's start time changes, flows arrive late, the past is declared void.  Every
    re-simulation must equal the oracle run that had the change from t = 0 -- whose own rollback is pinned against
    fresh runs -- and it must continue from the newest snapshot before the change, not from t = 0."""
    for w in (W.cfg1(batch=3, n_hosts=8, gph=4, n_leaves=4, n_spines=2), W.train_step(batch=2, n_hosts=4, gph=4, layers=2, buckets=2)):
        i = w.batch - 1
        inst = w.instances[i]
        base = oracle_run(w.desc, inst, mode=orc.MODE_FAST, base_seed=w.base_seed)
        t_ref = base.completion_times()
        t_end = t_ref.max()
        off, pr = base.preds()
        rel = np.array([t_ref[pr[off[f]:off[f + 1]]].max() if off[f + 1] > off[f] else 0.0 for f in range(base.num_flows)])
        flow = int(np.flatnonzero((rel > 0.45 * t_end) & (rel < 0.58 * t_end))[0])
        sim = B.Sim.from_workload(w, path=path)
        B.phs_set_snapshots(sim.h, 8)
        for frac in (0.2, 0.4, 0.6, 0.8):
            sim.run(until=frac * t_end)
        # (1) start-time update of a flow released between the snapshots at 0.4 and 0.6
        B.phs_update_flow_start(sim.h, i, flow, 0.9 * t_end)
        with pytest.raises(B.PhsError) as e:
            sim.completion_times(i)
        assert e.value.code == B.PHS_ESTATE
        sim.run()
        c = sim.counters()
        assert c["resumed_from_s"] == 0.4 * t_end and c["resumed_units"] > 0, c
        fresh = oracle_build(w.desc, inst, base_seed=w.base_seed)
        fresh.update_flow_start(flow, 0.9 * t_end)
        fresh.run(mode=orc.MODE_FAST)
        assert not np.array_equal(fresh.completion_times(), t_ref)
        assert_instance_matches(sim, i, fresh, check_log=False)
        for j in range(w.batch - 1):                     # the other instances are untouched
            assert_instance_matches(sim, j, oracle_run(w.desc, w.instances[j], mode=orc.MODE_FAST, base_seed=w.base_seed),
                                    check_log=False)
        # (2) the past declared void from 0.5 t_end: continue from the snapshot at 0.4, stop at 0.7
        B.phs_rollback(sim.h, 0.5 * t_end)
        sim.run(until=0.7 * t_end)
        assert sim.counters()["resumed_from_s"] == 0.4 * t_end
        part = oracle_build(w.desc, inst, base_seed=w.base_seed)
        part.update_flow_start(flow, 0.9 * t_end)
        part.run(mode=orc.MODE_FAST, until=0.7 * t_end)
        assert np.array_equal(sim.completion_times(i), part.completion_times(), equal_nan=True)
        assert np.array_equal(sim.bottlenecks(i), part.bottlenecks())
        # (3) garbage collection keeps what a rollback to >= the watermark needs
        B.phs_gc(sim.h, 0.45 * t_end)
        B.phs_rollback(sim.h, 0.45 * t_end)
        sim.run()
        assert sim.counters()["resumed_from_s"] == 0.4 * t_end
        assert_instance_matches(sim, i, fresh, check_log=False)
        # (4) a late submission (flows with an earlier timestamp, one of them behind an old flow) and the start time
        # of a flow without predecessors: tables rebuilt, results those of a fresh run
        late = (np.array([0, 1], np.int32), np.array([5, 6], np.int32), np.array([3e6, 5e5]),
                np.array([0.3, 0.05]) * t_end, np.array([0, 1, 1], np.int64), np.array([flow], np.int64))
        B.phs_add_flows(sim.h, i, *late)
        first_flow = int(np.flatnonzero(np.diff(off) == 0)[0])
        B.phs_update_flow_start(sim.h, i, first_flow, 0.01 * t_end)
        sim.run()
        assert sim.counters()["resumed_from_s"] == 0.0
        fresh.add_flows(*late)
        fresh.update_flow_start(first_flow, 0.01 * t_end)
        fresh.run(mode=orc.MODE_FAST)
        assert_instance_matches(sim, i, fresh, check_log=False)
        sim.close()


def test_multi_device_handle_shards_the_batch():
    """NEXT-4 / SURVEY.md 8(e): a handle bound to several devices cuts the batch into blocks of instances, one child
    handle per device, no data-path collective.  One GPU is visible here, so it is listed three times: three shards,
    three host threads, three sets of tables -- same results as the unsharded handle and the oracle."""
    import torch
    w = W.cfg3(batch=7)
    ref = B.Sim.from_workload(w)
    ref.run()
    sim = B.Sim.from_workload(w)
    B.phs_set_devices(sim.h, [0, 0, 0])
    B.phs_set_snapshots(sim.h, 4)
    sim.run()
    assert [B.phs_instance_device(sim.h, i) for i in range(7)] == [0] * 7
    for i in range(7):
        assert np.array_equal(sim.completion_times(i), ref.completion_times(i))
        assert np.array_equal(sim.bottlenecks(i), ref.bottlenecks(i))
        assert np.array_equal(sim.collective_times(i), ref.collective_times(i))
        assert sim.path_of(i) == ref.path_of(i)
    for i in (0, 3, 6):                                  # first, middle and last block: seeds follow the instance index
        assert_instance_matches(sim, i, oracle_run(w.desc, w.instances[i], mode=orc.MODE_FAST), check_log=False)
    assert np.array_equal(B.phs_get_all_completion_times(sim.h), B.phs_get_all_completion_times(ref.h))
    assert np.array_equal(B.phs_get_all_bottlenecks(sim.h), B.phs_get_all_bottlenecks(ref.h))
    c, cr = sim.counters(), ref.counters()
    assert c["n_events"] == cr["n_events"] and c["n_flow_events"] == cr["n_flow_events"] and c["sum_active"] == cr["sum_active"]
    out = torch.empty(sim.num_flows(5), dtype=torch.float64, device="cuda")
    B.phs_get_completion_times(sim.h, 5, device_ptr=out.data_ptr())
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), ref.completion_times(5))
    with pytest.raises(B.PhsError) as e:                 # late submissions are a single-device feature
        B.phs_add_flows(sim.h, 0, [0], [9], [1e6])
    assert e.value.code == B.PHS_ESTATE
    # stop times, rollback and start-time updates are routed to the shards
    t_end = max(ref.completion_times(i).max() for i in range(7))
    for frac in (0.3, 0.6):
        sim.run(until=frac * t_end)
        ref.run(until=frac * t_end)
        for i in range(7):
            assert np.array_equal(sim.completion_times(i), ref.completion_times(i), equal_nan=True)
    base = oracle_run(w.desc, w.instances[4], mode=orc.MODE_FAST)
    off, pr = base.preds()
    t4 = base.completion_times()
    rel = np.array([t4[pr[off[f]:off[f + 1]]].max() if off[f + 1] > off[f] else 0.0 for f in range(base.num_flows)])
    flow = int(np.flatnonzero((rel > 0.3 * t4.max()) & (rel < 0.7 * t4.max()))[0])
    B.phs_update_flow_start(sim.h, 4, flow, 0.9 * t_end)
    sim.run()
    fresh = oracle_build(w.desc, w.instances[4])
    fresh.update_flow_start(flow, 0.9 * t_end)
    fresh.run(mode=orc.MODE_FAST)
    assert_instance_matches(sim, 4, fresh, check_log=False)
    assert_instance_matches(sim, 2, oracle_run(w.desc, w.instances[2], mode=orc.MODE_FAST), check_log=False)
    sim.close(); ref.close()
