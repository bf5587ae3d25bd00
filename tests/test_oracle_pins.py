"""Pins of the CPU oracle against what the mathematics fixes.

None of these re-types the oracle's own formula: each expected value is a closed form, an iff-certificate,
a brute-force enumeration, a published test vector, or an invariance.

Mutants these pins are required to kill (tests/test_oracle_mutants.py applies each to a scratch copy of
oracle/orc_netsim.c and demands that at least one test of this file fails):
  M1  a released flow ignores its own start time            (st = now)                  -> test_p1_dependent_flow_...
  M2  the Q11 clamp removed from the settle step                                          -> test_q11_settle_clamp...
  M3  work counter sum_Lam doubled                                                        -> test_work_counters_...
  M4  leaf-spine down lane taken from the LOW hash bits instead of H >> 32                -> test_routing_leaf_spine_down_lane...
  M5  the FIFO predecessor (s-1, i) dropped                                               -> test_ring_dag_structure
  M6  `after` edge "received by rho" dropped                                              -> test_after_chains_...
  M7  argmin tie-break to the HIGHEST link id                                             -> test_p1 / test_p3
  M8  latency not added on release                                                        -> test_input_validation / P2
  M9  ring-after-all-to-all: edges to rho dropped                                         -> test_mixed_kind_after_edges_...
  M10 work counter sum_R counts events instead of iterations                              -> test_work_counters_...
"""
import itertools
import os

import numpy as np
import pytest

from oracle import orc
from paper_2505_01616_b200 import workloads as W
from util import completion_order, oracle_run

GOLD = os.path.join(os.path.dirname(__file__), "golden")
MiB = 2.0 ** 20
GiB = 2.0 ** 30


def golden(name):
    out = {}
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split("=")
                out[k.strip()] = float(v)
    return out


def single(n_hosts=2, gph=8, lat=1e-6, **kw):
    return W.topo_desc(W.TOPO_SINGLE, n_hosts, gph, hop_latency_s=lat, **kw)


def run_flows(desc, src, dst, nbytes, seed=0, **kw):
    inst = W.Instance(seed=seed, ops=[W.RawFlows(np.array(src, np.int32), np.array(dst, np.int32),
                                                 np.array(nbytes, np.float64), **kw)])
    return oracle_run(desc, inst)


# ------------------------------------------------------------------------------------------------ S2 hash
def test_splitmix64_published_vectors():
    # SplitMix64 (Steele, Lea, Flood 2014) from state 0: first three outputs of the public-domain reference.
    g = 0x9E3779B97F4A7C15
    assert orc.mix64(0) == 0xE220A8397B1DCDAF
    assert orc.mix64(g) == 0x6E789E6AA1B965F4
    assert orc.mix64((2 * g) & (2 ** 64 - 1)) == 0x06C45D188009454F


# ------------------------------------------------------------------------------------------------ S1 numbering
@pytest.mark.parametrize("wl,n_links", [(W.cfg0, 64), (lambda: W.cfg1(batch=1), 528), (W.cfg2, 7168),
                                        (lambda: W.cfg3(batch=1), 264), (lambda: W.cfg4(batch=1), 1152)])
def test_link_counts(wl, n_links):
    w = wl()
    assert orc.Sim(w.desc, 0).num_links == n_links


def test_flow_counts():
    assert sum(W.n_flows_of(o) for o in W.cfg0().instances[0].ops) == 480
    assert sum(W.n_flows_of(o) for o in W.cfg1(batch=1).instances[0].ops) == 5632
    assert sum(W.n_flows_of(o) for o in W.cfg2().instances[0].ops) == 1069056
    assert sum(W.n_flows_of(o) for o in W.cfg3(batch=1).instances[0].ops) == 7168
    assert sum(W.n_flows_of(o) for o in W.cfg4(batch=1).instances[0].ops) == 65280


# ------------------------------------------------------------------------------------------------ P1 lone flow
def test_p1_lone_flow_closed_form():
    g = golden("closed_forms.txt")
    d = single()
    s = run_flows(d, [0], [3], [4 * MiB])          # same host: NVLink up + NVLink down
    assert s.completion_times()[0] == pytest.approx(2e-6 + 4194304 / 450e9, rel=1e-12)
    assert s.completion_times()[0] == pytest.approx(g["p1_intra_host_4MiB"], rel=1e-9)
    assert list(s.paths()[1]) == [0, 7]
    s = run_flows(d, [0], [9], [4 * MiB])          # other host: NIC up + NIC down
    assert s.completion_times()[0] == pytest.approx(2e-6 + 4194304 / 50e9, rel=1e-12)
    assert s.completion_times()[0] == pytest.approx(g["p1_inter_host_4MiB"], rel=1e-9)
    assert list(s.paths()[1]) == [32 + 0, 32 + 19]
    assert list(s.bottlenecks()) == [32]           # tie between the two 50 GB/s links -> lowest id


def test_p1_lone_flow_start_time_and_fabric_bottleneck():
    # leaf-spine, cross-leaf: 4 hops; fabric slower than NIC -> fabric up link is the bottleneck (lower id than down)
    d = W.topo_desc(W.TOPO_LEAF_SPINE, 4, 2, nic_Bps=50e9, fabric_Bps=10e9, n_leaves=2, n_spines=2,
                    uplinks_per_leaf_spine=1, hop_latency_s=3e-6)
    s = run_flows(d, [0], [7], [1e6], start=np.array([5e-3]))
    off, links = s.paths()
    assert off[1] == 4
    assert s.completion_times()[0] == pytest.approx(5e-3 + 4 * 3e-6 + 1e6 / 10e9, rel=1e-12)
    assert s.bottlenecks()[0] == links[1]
    # fat tree cross-pod: 6 hops
    d = W.topo_desc(W.TOPO_FAT_TREE, 8, 2, fabric_Bps=25e9, k=4, agg_uplinks=2)
    s = run_flows(d, [0], [15], [1e6])
    assert s.paths()[0][1] == 6
    assert s.completion_times()[0] == pytest.approx(6e-6 + 1e6 / 25e9, rel=1e-12)


def test_p1_dependent_flow_waits_for_its_own_start_time():
    """SURVEY.md 8(c) S4 step 5 / PAPER.md L104 ("flows ... with the appropriate timestamps"): a released flow becomes
    active at max(start, t_pred) + Lat.  Closed form for a two-flow chain on link-disjoint pairs:
    t1 = max(start1, t0) + Lat + bytes1 / B, for start1 later than, equal to and earlier than t0."""
    d = single()
    B, Lat = 450e9, 2e-6
    t0 = Lat + 4e6 / B
    for start1 in (5 * t0, t0, 0.25 * t0, 0.0):
        s = run_flows(d, [0, 2], [1, 3], [4e6, 9e6], start=np.array([0.0, start1]),
                      dep_off=np.array([0, 0, 1]), dep_ids=np.array([0]))
        t = s.completion_times()
        assert t[0] == pytest.approx(t0, rel=1e-12)
        assert t[1] == pytest.approx(max(start1, t0) + Lat + 9e6 / B, rel=1e-12)
    # the same through a collective: step-0 flows of a ring chained `after` another one, with a later start time
    s = orc.Sim(single(n_hosts=1, gph=8), 0)
    a = s.add_collective(orc.ALLGATHER_RING, np.arange(4, dtype=np.int32), 4e6)
    T = 3 * (Lat + 1e6 / B)
    s.add_collective(orc.ALLGATHER_RING, np.arange(4, dtype=np.int32), 4e6, start=10 * T, after=[a])
    s.run()
    assert list(s.collective_times()) == pytest.approx([T, 10 * T + T], rel=1e-12)


def test_q11_settle_clamp_and_time_never_runs_backwards():
    """rem = max(rem - rate*dt, 0).  The step is pinned on its own (mul, sub, clamp), and
    through the property it protects: the clock of a run never goes backwards and no completion precedes its
    activation, on a workload full of near-simultaneous completions."""
    assert orc.settle(10.0, 2.0, 3.0) == 4.0
    assert orc.settle(1.0, 1e9, 1.0) == 0.0                      # drained more than it holds: clamped, not negative
    assert orc.settle(5e-324, 1.0, 1.0) == 0.0
    assert orc.settle(3.0, 0.5, 0.0) == 3.0
    d = single(lat=0.0, nic_Bps=1e9)
    rng = np.random.default_rng(11)
    base = np.floor(rng.uniform(1e5, 1e6, 40))
    sizes = np.concatenate([base, np.nextafter(base, np.inf), base + 2.0 ** -20])    # clusters of almost-equal sizes
    s = run_flows(d, list(rng.integers(0, 8, len(sizes))), [8 + i % 4 for i in range(len(sizes))], sizes)
    ev = s.event_log()
    assert np.all(np.diff(ev["t"]) >= 0)
    assert np.all(s.completion_times() > 0) and not np.isnan(s.completion_times()).any()


def test_work_counters_against_hand_counts():
    """orc_get_work_counters feeds the roofline's algorithmic bytes, so it is pinned against counts
    made by hand.  P6 (three flows, one shared link, zero latency): iteration 1 has A=3 on 4 links, one filling
    iteration; then A=2 on 3 links, A=1 on 2 links."""
    d = single(lat=0.0, nic_Bps=1e9)
    s = run_flows(d, [0, 1, 2], [8, 8, 8], [1e6, 2e6, 4e6])
    wk = s.work_counters()
    assert wk == {"sum_A": 6.0, "sum_Ah": 12.0, "sum_R": 3.0, "sum_LamR": 9.0, "sum_Lam": 9.0, "completions": 3.0,
                  "events": 3.0}
    # P7-like: A on two links, B, C on one each: 2 filling iterations on 5 links (3 NIC-up + 2 NIC-down)
    d = single(lat=0.0, nic_Bps=1e9)
    s = run_flows(d, [0, 1, 2], [8, 8, 9], [1e6, 1e6, 1e6])      # flows 0,1 share NIC-down(8); flow 2 alone
    wk = s.work_counters()
    # iteration 1: A=3, links {up0, up1, up2, dn8, dn9} = 5; bottleneck dn8 (0.5e9 each), then flow 2 (tie up2 / dn9): 2
    # flow 2 finishes at 1 ms, flows 0,1 at 2 ms: iteration 2: A=2, links 3, one filling iteration
    assert wk["sum_A"] == 5 and wk["sum_Ah"] == 10 and wk["sum_R"] == 3 and wk["sum_Lam"] == 8
    assert wk["sum_LamR"] == 5 * 2 + 3 * 1 and wk["completions"] == 3 and wk["events"] == 2
    # cfg0: no link is shared, so per event Lambda_act = 2A (two links per flow) and every flow is its own filling
    # iteration (R = A); the max-plus recurrence (P3) gives every activation and completion time, hence the events
    w = W.cfg0()
    o = oracle_run(w.desc, w.instances[0])
    T = maxplus_ring(np.arange(16), 30, 64 * MiB / 16, lambda i: 50e9 if i in (7, 15) else 450e9, 2e-6)
    dur = np.array([(64 * MiB / 16) / (50e9 if i in (7, 15) else 450e9) for i in range(16)])
    act = T - dur[None, :]                       # a flow is ACTIVE from T - chunk/B to T
    times = np.sort(np.concatenate([act.ravel(), T.ravel()]))
    events = [times[0]]
    for x in times[1:]:                          # distinct times (the recurrence is exact up to rounding)
        if x - events[-1] > 1e-12 * x:
            events.append(x)
    events = np.array(events)
    # flow f is counted in every iteration whose interval (e_{k-1}, e_k] lies inside (act_f, T_f]
    spans = np.searchsorted(events, T.ravel() * (1 + 1e-12)) - np.searchsorted(events, act.ravel() * (1 + 1e-12))
    wk = o.work_counters()
    assert wk["events"] == len(events) and wk["completions"] == 480
    assert wk["sum_A"] == spans.sum() and wk["sum_Ah"] == 2 * spans.sum() and wk["sum_Lam"] == 2 * spans.sum()
    assert wk["sum_R"] == spans.sum()
    # per-event A from the same intervals -> sum of A * 2A
    A_e = np.array([np.sum((act.ravel() < e * (1 - 1e-12)) & (T.ravel() >= e * (1 - 1e-12))) for e in events])
    assert wk["sum_LamR"] == np.sum(2 * A_e * A_e)


def test_comparison_modes_agree_within_the_stated_tolerance():
    """DESIGN.md sec 2 replaces two readings of SURVEY.md 8(c): R-LZ (settle a flow only when its rate changes) for
    S4.4 (debit every active flow at every event), and R-FX (integer rate quanta) for binary64 shares.  BASELINE.json
    states 1e-9 relative on completion times: the oracle keeps both original readings as modes (orc_run_ex flags) and
    they must agree with the default within that tolerance on the shrunken configs."""
    for w in (W.cfg1(batch=2, n_hosts=8, gph=4, n_leaves=4, n_spines=2), W.cfg2(k=4, agg_uplinks=1), W.cfg3(batch=2),
              W.cfg4(batch=1, n_hosts=8, gph=4, n_leaves=4, n_spines=2)):
        inst = w.instances[-1]
        ref = oracle_run(w.desc, inst).completion_times()
        for flags in (orc.FLAG_SETTLE_EVERY_EVENT, orc.FLAG_F64_SHARES, orc.FLAG_SETTLE_EVERY_EVENT | orc.FLAG_F64_SHARES):
            from util import oracle_build
            o = oracle_build(w.desc, inst)
            o.run(flags=flags)
            np.testing.assert_allclose(o.completion_times(), ref, rtol=1e-9, atol=0)
            assert not np.array_equal(o.completion_times(), ref) or flags == orc.FLAG_F64_SHARES   # the modes are live


# ------------------------------------------------------------------------------------------------ P2 uniform ring
@pytest.mark.parametrize("kind,steps", [(W.ALLREDUCE_RING, 14), (W.ALLGATHER_RING, 7), (W.REDUCESCATTER_RING, 7)])
def test_p2_uniform_ring(kind, steps):
    d = single()
    inst = W.Instance(seed=0, ops=[W.Coll(kind, np.arange(8, dtype=np.int32), 1 * GiB)])
    s = oracle_run(d, inst)
    expect = steps * (2e-6 + (2.0 ** 30 / 8) / 450e9)
    assert s.collective_times()[0] == pytest.approx(expect, rel=1e-12)
    if kind == W.ALLREDUCE_RING:
        assert expect == pytest.approx(golden("closed_forms.txt")["p2_ring_ar_n8_1GiB"], rel=1e-9)
    assert s.num_flows == steps * 8
    # every step's 8 flows finish together
    t = s.completion_times().reshape(steps, 8)
    assert np.all(t == t[:, :1])


# ------------------------------------------------------------------------------------------------ P3 max-plus ring
def maxplus_ring(ranks, steps, chunk, cap_of_sender, lat):
    """T(s,i) = max(T(s-1,i), T(s-1,i-1)) + d_i, d_i = Lat_i + chunk / B_i (contention-free ring)."""
    N = len(ranks)
    d = np.array([lat + chunk / cap_of_sender(i) for i in range(N)])
    T = np.zeros((steps, N))
    T[0] = d
    for s in range(1, steps):
        for i in range(N):
            T[s, i] = max(T[s - 1, i], T[s - 1, (i - 1) % N]) + d[i]
    return T


def test_p3_cfg0_maxplus_recurrence():
    w = W.cfg0()
    s = oracle_run(w.desc, w.instances[0])
    t = s.completion_times().reshape(30, 16)
    # senders 7 and 15 cross hosts (NIC, 50 GB/s), the others stay on NVLink (450 GB/s)
    T = maxplus_ring(np.arange(16), 30, 64 * MiB / 16, lambda i: 50e9 if i in (7, 15) else 450e9, 2e-6)
    np.testing.assert_allclose(t, T, rtol=1e-11, atol=0)
    g = golden("closed_forms.txt")
    assert t.max() == pytest.approx(g["p3_cfg0_makespan"], rel=1e-9)
    assert t[29, 8] == pytest.approx(g["p3_cfg0_T_29_8"], rel=1e-9)
    assert t[29, 0] == pytest.approx(g["p3_cfg0_T_29_8"], rel=1e-9)
    # no contention: both links of a path have equal capacity -> tie -> bneck is the lower link id
    off, links = s.paths()
    assert np.array_equal(s.bottlenecks(), np.minimum(links[off[:-1]], links[off[:-1] + 1]))


def test_p3_heterogeneous_ring_on_sweep_capacities():
    # one DP ring over 8 hosts with per-link random capacities (cfg3-style), contention-free -> recurrence
    w = W.cfg3(batch=1)
    inst = w.instances[0]
    inst.ops = [W.Coll(W.ALLREDUCE_RING, np.arange(0, 64, 8, dtype=np.int32), 64 * MiB)]
    s = oracle_run(w.desc, inst)
    cap = s.link_capacities()
    off, links = s.paths()
    lat = s.flows()[3]
    N = 8
    d = np.array([lat[i] + (64 * MiB / N) / cap[links[off[i]:off[i + 1]]].min() for i in range(N)])
    T = np.zeros((14, N))
    T[0] = d
    for st in range(1, 14):
        for i in range(N):
            T[st, i] = max(T[st - 1, i], T[st - 1, (i - 1) % N]) + d[i]
    # rates sit on a 2^-20 B/s grid: relative error <= 2^-20 / 1.25e10 per flow, far below 1e-11
    np.testing.assert_allclose(s.completion_times().reshape(14, N), T, rtol=1e-11)


# ------------------------------------------------------------------------------------------------ P4 certificate
def check_certificate(cap, path_off, path, flows, rate, bneck, n_links):
    """Bertsekas-Gallager: feasible AND every flow has a saturated link on which its rate is maximal  <=>  max-min
    fair.  Rates are floor-quantised to 2^-20 B/s, so a bottleneck may be short of capacity by < n_l quanta."""
    load = np.zeros(n_links)
    cnt = np.zeros(n_links, dtype=np.int64)
    mx = np.zeros(n_links)
    for f, r in zip(flows, rate):
        ls = path[path_off[f]:path_off[f + 1]]
        load[ls] += r
        cnt[ls] += 1
        mx[ls] = np.maximum(mx[ls], r)
    q = 2.0 ** -20
    assert np.all(load <= cap * (1 + 1e-12)), "link over capacity"
    for f, r, b in zip(flows, rate, bneck):
        ls = path[path_off[f]:path_off[f + 1]]
        assert b in ls
        ok = (load[ls] >= cap[ls] * (1 - 1e-12) - cnt[ls] * q) & (r >= mx[ls] * (1 - 1e-12) - q)
        assert ok.any(), f"flow {f} has no saturated link on which it is maximal"
        i = list(ls).index(b)
        assert ok[i], f"reported bottleneck {b} of flow {f} is not one"


@pytest.mark.parametrize("seed", range(6))
def test_p4_random_instances_certificate(seed):
    rng = np.random.default_rng(seed)
    n_links = int(rng.integers(3, 40))
    n_flows = int(rng.integers(1, 120))
    cap = np.floor(rng.uniform(1e9, 4e11, n_links))
    if seed % 2:
        cap[:] = 50e9                      # equal capacities: exact ties everywhere
    lens = rng.integers(1, min(6, n_links) + 1, n_flows)
    path_off = np.concatenate([[0], np.cumsum(lens)])
    path = np.concatenate([rng.choice(n_links, int(h), replace=False) for h in lens]).astype(np.int32)
    for mode in (orc.MODE_NAIVE, orc.MODE_FAST):
        rate, bneck, R, fb = orc.maxmin(cap, path_off, path, mode)
        check_certificate(cap, path_off, path, np.arange(n_flows), rate, bneck, n_links)
        assert 1 <= R <= n_links
        assert fb == bneck[np.argmin(rate)] or rate[bneck == fb].min() == rate.min()


@pytest.mark.parametrize("seed", range(8))
def test_removing_flows_leaves_the_slower_part_of_the_allocation_alone(seed):
    """The property the kernels' incremental re-solve rests on, checked on the ORACLE's from-scratch
    solves: remove flows from an allocation; every remaining flow whose old rate is below the smallest removed rate
    keeps its rate and its bottleneck, bit for bit.  (One-bottleneck-per-iteration filling picks links in ascending
    (share, id) order and its iterations before a removed flow's own bottleneck do not see the removal.)  Equal
    capacities in half of the cases: ties everywhere."""
    rng = np.random.default_rng(100 + seed)
    n_links = int(rng.integers(4, 40))
    n_flows = int(rng.integers(5, 160))
    cap = np.floor(rng.uniform(1e9, 4e11, n_links))
    if seed % 2:
        cap[:] = 50e9
    lens = rng.integers(1, min(6, n_links) + 1, n_flows)
    paths = [rng.choice(n_links, int(h), replace=False).astype(np.int32) for h in lens]

    def solve(keep):
        off = np.concatenate([[0], np.cumsum([len(paths[f]) for f in keep])])
        pth = np.concatenate([paths[f] for f in keep]).astype(np.int32)
        rate, bneck, _, _ = orc.maxmin(cap, off, pth, orc.MODE_FAST)
        return dict(zip(keep, rate)), dict(zip(keep, bneck))

    alive = list(range(n_flows))
    rate, bneck = solve(alive)
    unchanged_total = 0
    while len(alive) > 2:
        gone = [int(x) for x in rng.choice(alive, int(rng.integers(1, 4)), replace=False)]
        r_min = min(rate[f] for f in gone)
        alive = [f for f in alive if f not in gone]
        new_rate, new_bneck = solve(alive)
        for f in alive:
            if rate[f] < r_min:
                assert new_rate[f] == rate[f] and new_bneck[f] == bneck[f], (f, rate[f], r_min)
                unchanged_total += 1
            assert new_rate[f] >= rate[f] or rate[f] >= r_min          # nobody below the limit loses either
        rate, bneck = new_rate, new_bneck
    assert unchanged_total > 0 or n_flows < 8


@pytest.mark.parametrize("seed", range(8))
def test_adding_flows_leaves_the_slowest_part_of_the_allocation_alone(seed):
    """The other half of the incremental re-solve: add flows to an allocation; every old flow whose
    rate is below s* = min over the links of the added flows of floor(cap / n_new), n_new the link's flow count with the
    added flows, keeps its rate and its bottleneck, bit for bit.  (A link that carries an added flow has a share of at
    least s* throughout the new run, so the iterations of the old run below s* are picked again, in the same order.)
    Combined with removals in the same step: the limit is the smaller of the two."""
    rng = np.random.default_rng(300 + seed)
    n_links = int(rng.integers(4, 40))
    n_flows = int(rng.integers(20, 200))
    cap = np.floor(rng.uniform(1e9, 4e11, n_links))
    if seed % 2:
        cap[:] = 50e9
    capq = np.floor(cap * 2.0 ** 20)                    # exact in binary64 for these magnitudes
    lens = rng.integers(1, min(6, n_links) + 1, n_flows)
    paths = [rng.choice(n_links, int(h), replace=False).astype(np.int32) for h in lens]

    def solve(keep):
        off = np.concatenate([[0], np.cumsum([len(paths[f]) for f in keep])])
        pth = np.concatenate([paths[f] for f in keep]).astype(np.int32)
        rate, bneck, _, _ = orc.maxmin(cap, off, pth, orc.MODE_FAST)
        return dict(zip(keep, rate)), dict(zip(keep, bneck))

    alive = list(range(n_flows // 3))
    waiting = list(range(n_flows // 3, n_flows))
    rate, bneck = solve(alive)
    kept = 0
    while waiting:
        k = int(rng.integers(1, 4))
        new, waiting = waiting[:k], waiting[k:]
        gone = [int(x) for x in rng.choice(alive, int(rng.integers(0, 3)), replace=False)] if len(alive) > 4 else []
        alive2 = [f for f in alive if f not in gone] + new
        cnt = np.zeros(n_links)
        for f in alive2:
            cnt[paths[f]] += 1
        s_star = min(int(capq[l]) // int(cnt[l]) for f in new for l in paths[f]) * 2.0 ** -20   # exact integers
        limit = min([s_star] + [rate[f] for f in gone])
        new_rate, new_bneck = solve(alive2)
        for f in alive2:
            if f in rate and rate[f] < limit:
                assert new_rate[f] == rate[f] and new_bneck[f] == bneck[f], (f, rate[f], limit)
                kept += 1
        alive, rate, bneck = alive2, new_rate, new_bneck
    assert kept > 0


def test_p4_certificate_along_event_loop():
    # a contended mid-size run: shrunken cfg1 (DP rings share 2 uplinks per leaf) -- check EVERY recompute
    w = W.cfg1(batch=3, n_hosts=8, gph=4, n_leaves=4, n_spines=2)
    for inst in w.instances[1:]:
        s = oracle_run(w.desc, inst, trace=True)
        ev, fl, rate, t0, t1 = s.trace()
        off, links = s.paths()
        cap = s.link_capacities()
        bn = s.bottlenecks()
        cuts = np.flatnonzero(np.diff(ev)) + 1
        n_checked = 0
        for idx in np.split(np.arange(len(ev)), cuts)[::7]:
            # bneck[] holds the LAST bottleneck of each flow; only check membership for flows of the final events
            load = np.zeros(len(cap)); mx = np.zeros(len(cap)); cnt = np.zeros(len(cap))
            for f, r in zip(fl[idx], rate[idx]):
                ls = links[off[f]:off[f + 1]]
                load[ls] += r; cnt[ls] += 1; mx[ls] = np.maximum(mx[ls], r)
            assert np.all(load <= cap * (1 + 1e-12))
            for f, r in zip(fl[idx], rate[idx]):
                ls = links[off[f]:off[f + 1]]
                ok = (load[ls] >= cap[ls] * (1 - 1e-12) - cnt[ls] * 2.0 ** -20) & (r >= mx[ls] * (1 - 1e-12) - 2.0 ** -20)
                assert ok.any()
            n_checked += 1
        assert n_checked > 20
        assert np.all(bn >= 0)


# ------------------------------------------------------------------------------------------------ P5 brute force
def brute_force_maxmin(cap, paths, grid):
    """Lexicographically largest ascending-sorted feasible rate vector over rates in `grid` (exhaustive)."""
    F = len(paths)
    G = np.array(list(itertools.product(grid, repeat=F)), dtype=np.int64)
    ok = np.ones(len(G), dtype=bool)
    for l, c in enumerate(cap):
        on = [f for f in range(F) if l in paths[f]]
        if on:
            ok &= G[:, on].sum(axis=1) <= c
    G = G[ok]
    S = np.sort(G, axis=1)
    best = np.lexsort(tuple(S[:, j] for j in range(F - 1, -1, -1)))[-1]
    return G[best], S[best]


@pytest.mark.parametrize("seed", range(40))
def test_p5_brute_force_lexicographic_maxmin(seed):
    rng = np.random.default_rng(1000 + seed)
    n_links = int(rng.integers(1, 5))
    F = int(rng.integers(1, 4)) if seed % 8 else 4
    cap = rng.integers(1, 5, n_links) * 12                      # caps in {12,24,36,48}: every share is an integer
    paths = []
    for _ in range(F):
        h = int(rng.integers(1, n_links + 1))
        paths.append(sorted(rng.choice(n_links, h, replace=False).tolist()))
    grid = range(0, 49)
    best, best_sorted = brute_force_maxmin(cap, paths, grid)
    path_off = np.concatenate([[0], np.cumsum([len(p) for p in paths])])
    path = np.concatenate(paths).astype(np.int32)
    rate, bneck, R, fb = orc.maxmin(cap.astype(np.float64), path_off, path, orc.MODE_NAIVE)
    # the max-min allocation is unique -> the whole vector must match, not just the sorted one
    assert np.array_equal(rate, best.astype(np.float64))
    for f in range(F):
        assert bneck[f] in paths[f]


# ------------------------------------------------------------------------------------------------ P6 processor sharing
def test_p6_processor_sharing_closed_form():
    # three senders on host 0, one receiver on host 1: they share only the receiver's NIC-down link (C = 1e9 B/s)
    d = single(lat=0.0, nic_Bps=1e9)
    s = run_flows(d, [0, 1, 2], [8, 8, 8], [1e6, 2e6, 4e6])
    np.testing.assert_allclose(s.completion_times(), [3e-3, 5e-3, 7e-3], rtol=1e-11)
    # O3 = bottleneck in the LAST solve while active: flows 0,1 still share NIC-down(8)=49; flow 2 ends alone, and
    # alone its two equal-capacity links tie -> lowest id = NIC-up(2)=36
    assert list(s.bottlenecks()) == [49, 49, 36]
    # general n: t_k = t_{k-1} + (s_k - s_{k-1}) (n-k+1) / C
    rng = np.random.default_rng(5)
    sizes = np.sort(np.floor(rng.uniform(1e5, 1e7, 7)))
    s = run_flows(d, list(range(7)), [9] * 7, sizes)
    t, prev, tk = [], 0.0, 0.0
    for k, sz in enumerate(sizes):
        tk += (sz - prev) * (7 - k) / 1e9
        prev = sz
        t.append(tk)
    np.testing.assert_allclose(s.completion_times(), t, rtol=1e-11)


# ------------------------------------------------------------------------------------------------ P7 parking lot
def test_p7_parking_lot():
    c1, c2 = 30e9, 100e9
    cap = np.array([7e11, c1, c2])
    path_off = np.array([0, 2, 3, 4])
    path = np.array([1, 2, 1, 2], np.int32)            # A on links 1,2 ; B on 1 ; C on 2
    for mode in (orc.MODE_NAIVE, orc.MODE_FAST):
        rate, bneck, R, fb = orc.maxmin(cap, path_off, path, mode)
        np.testing.assert_allclose(rate, [c1 / 2, c1 / 2, c2 - c1 / 2], rtol=1e-15)
        assert list(bneck) == [1, 1, 2] and R == 2 and fb == 1


# ------------------------------------------------------------------------------------------------ P8 uniform all-to-all
@pytest.mark.parametrize("N", [9, 8])
def test_p8_uniform_alltoall_single_switch(N):
    B, S = 50e9, 64 * MiB
    d = single(n_hosts=N, gph=1)
    inst = W.Instance(seed=0, ops=[W.Coll(W.ALLTOALL, np.arange(N, dtype=np.int32), S)])
    s = oracle_run(d, inst)
    t = s.completion_times()
    assert len(t) == N * (N - 1)
    np.testing.assert_allclose(t, 2e-6 + (S / N) * (N - 1) / B, rtol=1e-12)
    ev = s.event_log()
    if N == 9:
        # B/(N-1) is exact on the 2^-20 B/s grid: every flow gets bit-equal rate -> ONE completion event
        assert np.all(t == t[0])
        assert ev["n_completed"].max() == N * (N - 1) and (ev["n_completed"] > 0).sum() == 1
    else:
        # B/7 is not on the grid: the floor remainder (< 7 quanta) goes to later-frozen flows, rates differ by
        # at most one quantum (2^-20 B/s) and completion times by a few ulp
        assert len(np.unique(t)) <= 4
    src, dst, b, lat = s.flows()
    assert np.array_equal(src, np.repeat(np.arange(N), N - 1))
    assert np.all(src != dst) and np.all(b == S / N)


# ------------------------------------------------------------------------------------------------ S3 DAG pins
def test_ring_dag_structure():
    N = 5
    d = single(n_hosts=1, gph=8)
    s = orc.Sim(d, 0)
    ranks = np.array([3, 0, 6, 1, 4], np.int32)
    s.add_collective(orc.ALLREDUCE_RING, ranks, 5e6)
    off, pr = s.preds()
    src, dst, b, lat = (None,) * 4
    s.run()
    src, dst, b, lat = s.flows()
    assert s.num_flows == 2 * (N - 1) * N
    for st in range(2 * (N - 1)):
        for i in range(N):
            f = st * N + i
            assert src[f] == ranks[i] and dst[f] == ranks[(i + 1) % N] and b[f] == 1e6
            p = sorted(pr[off[f]:off[f + 1]].tolist())
            if st == 0:
                assert p == []
            else:
                assert p == sorted([(st - 1) * N + (i - 1) % N, (st - 1) * N + i])


def test_after_chains_per_rank_not_global_barrier():
    d = single(n_hosts=1, gph=8)
    s = orc.Sim(d, 0)
    a = s.add_collective(orc.ALLREDUCE_RING, np.arange(4, dtype=np.int32), 4e6)          # ranks 0..3
    b = s.add_collective(orc.ALLGATHER_RING, np.array([2, 3, 4, 5], np.int32), 4e6, after=[a])
    off, pr = s.preds()
    fa, la = 0, 5 * 4                # A: 6 steps x 4; last step starts at flow 20
    fb = 6 * 4
    # B's step-0 flow i has sender [2,3,4,5][i]; ranks 2,3 are ring indices 2,3 of A; 4,5 are not in A
    assert sorted(pr[off[fb + 0]:off[fb + 1]]) == [la + 1, la + 2]       # sent by 2 = (5,2); received by 2 = (5,1)
    assert sorted(pr[off[fb + 1]:off[fb + 2]]) == [la + 2, la + 3]
    assert off[fb + 3] - off[fb + 2] == 0 and off[fb + 4] - off[fb + 3] == 0
    s.run()
    t = s.completion_times()
    step = 2e-6 + 1e6 / 450e9
    # ranks 4 and 5 start B's first step at t=0 (4->5 shares no link with A), ranks 2 and 3 only after A's last
    # step has left / reached them; B's 2->3 then runs uncontended (A's only possible straggler 3->0 is link-disjoint)
    assert t[fb + 2] == pytest.approx(step, rel=1e-12)
    assert t[fb + 0] == pytest.approx(max(t[la + 1], t[la + 2]) + step, rel=1e-12)
    assert t[fb + 0] > 6 * step


def test_chained_equals_concurrent_total_on_uniform_ring():
    # two identical ring all-reduces: chained -> 2 T ; also pins `after` on every rank
    d = single(n_hosts=1, gph=8)
    T = 14 * (2e-6 + (64 * MiB / 8) / 450e9)
    s = orc.Sim(d, 0)
    a = s.add_collective(orc.ALLREDUCE_RING, np.arange(8, dtype=np.int32), 64 * MiB)
    s.add_collective(orc.ALLREDUCE_RING, np.arange(8, dtype=np.int32), 64 * MiB, after=[a])
    s.run()
    assert list(s.collective_times()) == pytest.approx([T, 2 * T], rel=1e-12)
    # concurrent: the two rings share every link half/half; each step takes Lat + 2*chunk/B
    s = orc.Sim(d, 0)
    s.add_collective(orc.ALLREDUCE_RING, np.arange(8, dtype=np.int32), 64 * MiB)
    s.add_collective(orc.ALLREDUCE_RING, np.arange(8, dtype=np.int32), 64 * MiB)
    s.run()
    T2 = 14 * (2e-6 + 2 * (64 * MiB / 8) / 450e9)
    assert list(s.collective_times()) == pytest.approx([T2, T2], rel=1e-11)


def test_alltoall_after_alltoall_preds():
    d = single(n_hosts=1, gph=4)
    s = orc.Sim(d, 0)
    a = s.add_collective(orc.ALLTOALL, np.arange(4, dtype=np.int32), 4e6)
    s.add_collective(orc.ALLTOALL, np.arange(4, dtype=np.int32), 4e6, after=[a])
    off, pr = s.preds()
    src, dst = None, None
    s.run()
    src, dst, _, _ = s.flows()
    for f in range(12, 24):
        rho = src[f]
        want = sorted([g for g in range(12) if src[g] == rho or dst[g] == rho])
        assert sorted(pr[off[f]:off[f + 1]].tolist()) == want


def test_mixed_kind_after_edges_against_hand_written_lists():
    """S3 `after` between different collective kinds, against lists written out by hand (N = 3)."""
    d = single(n_hosts=1, gph=8)
    # all-to-all over [0,1,2]: flows 0:0->1 1:0->2 2:1->0 3:1->2 4:2->0 5:2->1 ; then a ring all-gather over [2,0,1]
    s = orc.Sim(d, 0)
    a = s.add_collective(orc.ALLTOALL, np.array([0, 1, 2], np.int32), 3e6)
    s.add_collective(orc.ALLGATHER_RING, np.array([2, 0, 1], np.int32), 3e6, after=[a])
    off, pr = s.preds()
    want = {6: [1, 3, 4, 5],      # sender 2: everything from / to rank 2
            7: [0, 1, 2, 4],      # sender 0
            8: [0, 2, 3, 5]}      # sender 1
    for f, p in want.items():
        assert sorted(pr[off[f]:off[f + 1]].tolist()) == p
    assert sorted(pr[off[9]:off[10]].tolist()) == [6, 8] and sorted(pr[off[10]:off[11]].tolist()) == [6, 7]
    # ring all-reduce over [1,2,3] (4 steps x 3; last step = flows 9,10,11: 1->2, 2->3, 3->1); then an all-to-all
    # over [0,1,2]: rank 0 is not in the ring (no edge), rank 1 sent 9 and received 11, rank 2 sent 10 and received 9
    s = orc.Sim(d, 0)
    a = s.add_collective(orc.ALLREDUCE_RING, np.array([1, 2, 3], np.int32), 3e6)
    s.add_collective(orc.ALLTOALL, np.array([0, 1, 2], np.int32), 3e6, after=[a])
    off, pr = s.preds()
    want = {12: [], 13: [], 14: [9, 11], 15: [9, 11], 16: [9, 10], 17: [9, 10]}
    for f, p in want.items():
        assert sorted(pr[off[f]:off[f + 1]].tolist()) == p


# ------------------------------------------------------------------------------------------------ NEXT-3 collectives
@pytest.mark.parametrize("kind", [W.BROADCAST_CHAIN, W.REDUCE_CHAIN])
@pytest.mark.parametrize("N,C", [(5, 4), (8, 1), (3, 7)])
def test_next3_pipelined_chain_closed_form(kind, N, C):
    """A chain of N ranks moving C chunks over link-disjoint hops is the max-plus recurrence
    T(c, i) = max(T(c, i-1), T(c-1, i)) + d, d = Lat + (bytes / C) / B: the last chunk leaves the last hop at
    (C + N - 2) d; flow (c, i) finishes at (c + i + 1) d."""
    d = single(n_hosts=1, gph=8)
    s = orc.Sim(d, 0)
    ranks = np.array([5, 2, 7, 0, 3, 6, 1, 4][:N], np.int32)
    s.add_collective(kind, ranks, 6e6, chunks=C)
    s.run()
    step = 2e-6 + (6e6 / C) / 450e9
    t = s.completion_times().reshape(C, N - 1)
    want = np.array([[(c + i + 1) * step for i in range(N - 1)] for c in range(C)])
    np.testing.assert_allclose(t, want, rtol=1e-12)
    assert s.collective_times()[0] == pytest.approx((C + N - 2) * step, rel=1e-12)
    src, dst, b, _ = s.flows()
    hops = [(ranks[i], ranks[i + 1]) if kind == W.BROADCAST_CHAIN else (ranks[N - 1 - i], ranks[N - 2 - i])
            for i in range(N - 1)]
    assert [(a, b_) for a, b_ in zip(src, dst)] == hops * C and np.all(b == 6e6 / C)


def test_next3_tree_allreduce_structure_and_closed_form():
    """Binary tree in heap order, hand-written for N = 4, C = 2: positions 0 <- 1, 2 ; 1 <- 3.  Per chunk: up(1), up(2),
    up(3), down(1), down(2), down(3).  Then the closed form of a perfect tree of 7 on one NVSwitch: the two children of
    a node share its down link on the way up and its up link on the way down, so each of the 4 levels takes
    Lat + 2 bytes / B."""
    d = single(n_hosts=1, gph=8)
    s = orc.Sim(d, 0)
    r = np.array([6, 1, 4, 3], np.int32)
    s.add_collective(orc.ALLREDUCE_TREE, r, 8e6, chunks=2)
    off, pr = s.preds()
    s.run()
    src, dst, b, _ = s.flows()
    edges = [(1, 6), (4, 6), (3, 1), (6, 1), (6, 4), (1, 3)]           # up(1) up(2) up(3) down(1) down(2) down(3)
    assert [(a, b_) for a, b_ in zip(src, dst)] == edges * 2 and np.all(b == 4e6)
    want = {0: [2], 1: [], 2: [], 3: [0, 1], 4: [0, 1], 5: [3],          # chunk 0
            6: [0, 8], 7: [1], 8: [2], 9: [3, 6, 7], 10: [4, 6, 7], 11: [5, 9]}
    for f, p in want.items():
        assert sorted(pr[off[f]:off[f + 1]].tolist()) == p, f
    s = orc.Sim(d, 0)
    s.add_collective(orc.ALLREDUCE_TREE, np.arange(7, dtype=np.int32), 4e6)
    s.run()
    assert s.collective_times()[0] == pytest.approx(4 * (2e-6 + 2 * 4e6 / 450e9), rel=1e-12)


def test_next3_after_edges_against_hand_written_lists():
    """`after` with the chain / tree kinds on either side (N = 3), lists written out by hand."""
    d = single(n_hosts=1, gph=8)
    # A = chain broadcast over [0,1,2], 2 chunks: flows 0:(c0) 0->1, 1:(c0) 1->2, 2:(c1) 0->1, 3:(c1) 1->2.
    # B = ring all-gather over [2,0,1] after A: sender 2 receives 3; sender 0 sends 2; sender 1 receives 2, sends 3
    s = orc.Sim(d, 0)
    a = s.add_collective(orc.BROADCAST_CHAIN, np.array([0, 1, 2], np.int32), 2e6, chunks=2)
    s.add_collective(orc.ALLGATHER_RING, np.array([2, 0, 1], np.int32), 3e6, after=[a])
    off, pr = s.preds()
    assert [sorted(pr[off[f]:off[f + 1]].tolist()) for f in (4, 5, 6)] == [[3], [2], [2, 3]]
    # A = ring reduce-scatter over [1,2,0] (2 steps x 3: last step = flows 3: 1->2, 4: 2->0, 5: 0->1);
    # B = tree all-reduce over [2,0,1] (up(1): 0->2, up(2): 1->2, down(1), down(2)) after A: the leaves' up flows wait:
    # sender 0 sent 5, received 4; sender 1 sent 3, received 5
    s = orc.Sim(d, 0)
    a = s.add_collective(orc.REDUCESCATTER_RING, np.array([1, 2, 0], np.int32), 3e6)
    s.add_collective(orc.ALLREDUCE_TREE, np.array([2, 0, 1], np.int32), 3e6, after=[a])
    off, pr = s.preds()
    assert [sorted(pr[off[f]:off[f + 1]].tolist()) for f in (6, 7, 8, 9)] == [[4, 5], [3, 5], [6, 7], [6, 7]]
    # A = tree over [0,1,2], 1 chunk: 0: up(1) 1->0, 1: up(2) 2->0, 2: down(1) 0->1, 3: down(2) 0->2; B = reduce chain
    # over [2,1] (hop 0: 1->2) after A: sender 1 sent 0, received 2
    s = orc.Sim(d, 0)
    a = s.add_collective(orc.ALLREDUCE_TREE, np.array([0, 1, 2], np.int32), 3e6)
    s.add_collective(orc.REDUCE_CHAIN, np.array([2, 1], np.int32), 3e6, after=[a], chunks=3)
    off, pr = s.preds()
    assert [sorted(pr[off[f]:off[f + 1]].tolist()) for f in (4, 5, 6)] == [[0, 2], [4], [5]]


# ------------------------------------------------------------------------------------------------ NEXT-2 compute spans
def test_next2_compute_spans_closed_forms():
    """Reading S7 (PAPER.md L84 / L94 / L106 / L206): a span alone on its lane ends at EXACTLY t_act + d (the 2^32
    scaling is exact in binary64); spans overlapping on one lane share it (processor sharing, P6); a collective
    chained behind compute is fully exposed (Dc + Tc), next to it fully overlapped (max)."""
    d = single(n_hosts=1, gph=8, compute_lanes=2)
    s = orc.Sim(d, 0)
    assert s.num_links == 32 + 16                                     # engine links follow the network links
    dur = [1e-3, 3.3e-4, 7e-5]
    s.add_spans([0, 5, 5], dur, lane=[0, 0, 1], start=[0.0, 1e-4, 2.5e-4])
    s.run()
    assert list(s.completion_times()) == [0.0 + dur[0], 1e-4 + dur[1], 2.5e-4 + dur[2]]          # bit-equal
    assert list(s.bottlenecks()) == [32 + 0, 32 + 5 * 2, 32 + 5 * 2 + 1]
    # two spans on ONE lane at the same time: each gets half the engine (P6 with C = 2^32): 2 d, then the longer alone
    s = orc.Sim(d, 0)
    s.add_spans([3, 3], [1e-4, 3e-4], lane=[1, 1])
    s.run()
    np.testing.assert_allclose(s.completion_times(), [2e-4, 4e-4], rtol=1e-12)
    # exposed: all-gather over ranks 0..3 behind a span on every rank; overlapped: the same side by side
    Tc = 3 * (2e-6 + 1e6 / 450e9)
    Dc = [2e-4, 5e-4, 1e-4, 3e-4]
    s = orc.Sim(d, 0)
    s.add_spans([0, 1, 2, 3], Dc)
    s.add_collective(orc.ALLGATHER_RING, np.arange(4, dtype=np.int32), 4e6, after_flows=[0, 1, 2, 3])
    last = s.add_spans([0], [1e-5], dep_off=[0, 2], dep_ids=[4 + 2 * 4 + 0, 4 + 2 * 4 + 3])     # rank 0's last send / receive
    s.run()
    t = s.completion_times()
    step = 2e-6 + 1e6 / 450e9
    # ring recurrence with staggered starts: T(0,i) = Dc[i] + step; T(s,i) = max(T(s-1,i), T(s-1,i-1)) + step
    T = np.zeros((3, 4)); T[0] = np.array(Dc) + step
    for st in range(1, 3):
        for i in range(4):
            T[st, i] = max(T[st - 1, i], T[st - 1, (i - 1) % 4]) + step
    np.testing.assert_allclose(t[4:16].reshape(3, 4), T, rtol=1e-12)
    assert t[last] == pytest.approx(max(T[2, 0], T[2, 3]) + 1e-5, rel=1e-12)
    assert s.collective_times()[0] > max(Dc) + Tc * 0.99                                       # exposed
    s = orc.Sim(d, 0)
    s.add_spans([0, 1, 2, 3], Dc)
    s.add_collective(orc.ALLGATHER_RING, np.arange(4, dtype=np.int32), 4e6)
    s.run()
    assert s.collective_times()[0] == pytest.approx(Tc, rel=1e-12)                             # overlapped
    with pytest.raises(orc.OrcError):
        orc.Sim(single(), 0).add_spans([0], [1e-3])                                            # no compute lanes


# ------------------------------------------------------------------------------------------------ NEXT-1 time rollback
def _same_results(a, b):
    assert np.array_equal(a.completion_times(), b.completion_times())
    assert np.array_equal(a.bottlenecks(), b.bottlenecks())
    assert np.array_equal(a.event_log(), b.event_log())
    for x, y in zip(a.history(), b.history()):
        assert np.array_equal(x, y)


def _rollback_workloads():
    yield W.cfg1(batch=2, n_hosts=8, gph=4, n_leaves=4, n_spines=2), 1
    yield W.train_step(batch=1, n_hosts=4, gph=4, layers=2, buckets=2), 0
    yield W.cfg4(batch=1, n_hosts=4, gph=4, n_leaves=2, n_spines=2), 0


def test_next1_advancing_in_steps_equals_one_run():
    """PAPER.md L167 "advancing the simulation ... up to a specified time", repeatedly: every call rebuilds the state
    from the throughput history (L128) and continues; the end result is the one-shot run, bit for bit."""
    from util import oracle_build
    for w, i in _rollback_workloads():
        ref = oracle_run(w.desc, w.instances[i])
        t_end = ref.completion_times().max()
        o = oracle_build(w.desc, w.instances[i])
        for frac in (0.0, 0.13, 0.13, 0.5, 0.77):
            o.run(until=frac * t_end)
            done = ref.completion_times() <= frac * t_end
            assert np.array_equal(o.completion_times()[done], ref.completion_times()[done])
            assert np.isnan(o.completion_times()[~done]).all()
        o.run()
        _same_results(o, ref)


def test_next1_rollback_and_rerun_equals_a_fresh_run():
    """The property that fixes the rollback (Fig. 4): after the simulator has run ahead to T1,
    changing a flow's start time (L167) or submitting flows with an earlier timestamp T2 rolls back to T2, and the
    re-simulation equals -- completion times, bottlenecks, event log, throughput history, all bit for bit -- a fresh
    run that had the change from t = 0.  T2 before, inside and after the lives of the affected flows."""
    from util import oracle_build
    rng = np.random.default_rng(9)
    for w, i in _rollback_workloads():
        inst = w.instances[i]
        base = oracle_run(w.desc, inst)
        t0 = base.completion_times()
        t_end = t0.max()
        F = base.num_flows
        mattered = 0
        for case in range(6):
            flows = rng.choice(F, 3, replace=False)
            T1 = [0.3, 0.6, 1.0, 0.9, 0.5, 2.0][case] * t_end          # how far the simulator ran ahead
            new_start = [0.1, 0.55, 0.2, 1.3, 0.0, 0.7][case] * t_end * np.array([1.0, 0.5, 1.1])
            late = W.RawFlows(np.array([0, 1], np.int32), np.array([5, 6], np.int32), np.array([3e6, 5e5]),
                              start=np.array([0.4, 0.05]) * t_end, dep_off=np.array([0, 1, 1], np.int64),
                              dep_ids=np.array([int(flows[0])], np.int64))
            fresh = oracle_build(w.desc, inst)                          # the change known from t = 0
            for f, st in zip(flows, new_start):
                fresh.update_flow_start(int(f), float(st))
            fresh.add_flows(late.src, late.dst, late.nbytes, late.start, late.dep_off, late.dep_ids)
            fresh.run()
            live = oracle_build(w.desc, inst)                           # the change arrives at T1
            live.run(until=T1)
            n_before = len(live.event_log())
            for f, st in zip(flows, new_start):
                live.update_flow_start(int(f), float(st))
            live.add_flows(late.src, late.dst, late.nbytes, late.start, late.dep_off, late.dep_ids)
            assert len(live.event_log()) <= n_before                   # rolled back (or nothing to roll back)
            live.run()
            _same_results(live, fresh)
            mattered += not np.array_equal(fresh.completion_times()[:F], t0)
        assert mattered >= 3                                             # the changes do move the old flows
    # an explicit rollback forgets the future and nothing else
    w, i = next(_rollback_workloads())
    ref = oracle_run(w.desc, w.instances[i])
    o = oracle_run(w.desc, w.instances[i])
    T = 0.4 * ref.completion_times().max()
    o.rollback(T)
    assert np.isnan(o.completion_times()[ref.completion_times() >= T]).all()
    assert np.array_equal(o.event_log(), ref.event_log()[ref.event_log()["t"] < T])
    o.run()
    _same_results(o, ref)
    T = float(ref.event_log()["t"][len(ref.event_log()) // 2])            # exactly an event time: that event goes too
    o.rollback(T)
    assert np.array_equal(o.event_log(), ref.event_log()[ref.event_log()["t"] < T])
    assert np.isnan(o.completion_times()[ref.completion_times() >= T]).all()
    o.run()
    _same_results(o, ref)


def test_next1_gc_keeps_every_later_rollback_exact():
    """history older than the watermark is dropped; results after GC(T) equal results without GC for
    every later rollback target >= T, and a rollback below T is refused."""
    from util import oracle_build
    w, i = next(_rollback_workloads())
    inst = w.instances[i]
    ref = oracle_run(w.desc, inst)
    t_end = ref.completion_times().max()
    n_hist = len(ref.history()[0])
    off, pr = ref.preds()
    t_ref = ref.completion_times()
    rel = np.array([t_ref[pr[off[f]:off[f + 1]]].max() if off[f + 1] > off[f] else 0.0 for f in range(ref.num_flows)])
    flow = int(np.flatnonzero((rel > 0.62 * t_end) & (rel < 0.75 * t_end))[0])     # released between the watermarks and T1
    for Tw, T2 in ((0.3, 0.7), (0.5, 0.9), (0.6, 0.78)):
        o = oracle_build(w.desc, inst)
        o.run(until=0.8 * t_end)
        o.gc(Tw * t_end)
        assert len(o.history()[0]) < n_hist
        with pytest.raises(orc.OrcError):
            o.rollback(0.5 * Tw * t_end)
        with pytest.raises(orc.OrcError):
            o.update_flow_start(0, 0.1 * t_end)          # a flow that started at t = 0: below the watermark
        o.update_flow_start(flow, T2 * t_end)
        assert len(o.event_log()) < len(ref.event_log()[ref.event_log()["t"] <= 0.8 * t_end])     # it did roll back
        o.run()
        fresh = oracle_build(w.desc, inst)
        fresh.update_flow_start(flow, T2 * t_end)
        fresh.run()
        assert not np.array_equal(fresh.completion_times(), t_ref)
        assert np.array_equal(o.completion_times(), fresh.completion_times())
        assert np.array_equal(o.bottlenecks(), fresh.bottlenecks())
        assert np.array_equal(o.event_log(), fresh.event_log())
        fo, to, ro = o.history()
        ff, tf, rf = fresh.history()
        keep = tf >= Tw * t_end                                           # what GC may not touch
        late = to >= Tw * t_end
        assert np.array_equal(fo[late], ff[keep]) and np.array_equal(to[late], tf[keep]) and np.array_equal(ro[late], rf[keep])


# ------------------------------------------------------------------------------------------------ NEXT-4 graph topologies
def _star(G, cap=50e9, lat=1e-6):
    lf, lt = [], []
    for g in range(G):
        lf += [g, G]; lt += [G, g]          # link 2g: GPU g -> switch, 2g+1: switch -> GPU g
    return W.graph_desc(G, G + 1, lf, lt, [cap] * (2 * G), [lat] * (2 * G))


def test_next4_graph_topology_closed_forms_and_structure():
    """Reading S8 (topology configuration as input): a user-supplied link list, shortest-path ECMP.
    (1) a line GPU0 - s - s - GPU1 with different capacities and latencies: t = sum(lat) + bytes / min(cap), and the
    bottleneck is the slowest link; (2) a star equals the single-switch preset on the NIC links, time for time;
    (3) in a two-spine fabric every path is a shortest path made of consecutive links, both spines are used about
    equally, and a connection keeps its path; (4) unroutable or too long pairs are refused."""
    d = W.graph_desc(2, 4, [0, 2, 3, 1, 3, 2], [2, 3, 1, 3, 2, 0], [40e9, 10e9, 25e9, 40e9, 10e9, 25e9],
                     [1e-6, 3e-6, 2e-6, 1e-6, 3e-6, 2e-6])
    s = orc.Sim(d, 0)
    s.add_flows([0, 1], [1, 0], [5e6, 2e6])
    s.run()
    assert list(s.paths()[1]) == [0, 1, 2, 3, 4, 5]
    assert s.completion_times()[0] == pytest.approx(6e-6 + 5e6 / 10e9, rel=1e-12)
    assert s.completion_times()[1] == pytest.approx(6e-6 + 2e6 / 10e9, rel=1e-12)
    assert list(s.bottlenecks()) == [1, 4]
    # (2) star == TOPO_SINGLE with one GPU per host (NIC links only), same workload
    ops = [W.Coll(W.ALLREDUCE_RING, np.arange(8, dtype=np.int32), 32 * MiB), W.Coll(W.ALLTOALL, np.arange(8, dtype=np.int32), 8 * MiB, 1e-4)]
    a = oracle_run(_star(8), W.Instance(seed=3, ops=ops))
    b = oracle_run(W.topo_desc(W.TOPO_SINGLE, 8, 1), W.Instance(seed=3, ops=ops))
    assert np.array_equal(a.completion_times(), b.completion_times())
    assert np.array_equal(a.bottlenecks() + 16, b.bottlenecks())          # the preset numbers its NIC links from 2G on
    # (3) 8 GPUs, 2 leaves (nodes 8, 9), 2 spines (10, 11)
    lf, lt = [], []
    for g in range(8):
        leaf = 8 + g // 4
        lf += [g, leaf]; lt += [leaf, g]
    for leaf in (8, 9):
        for sp in (10, 11):
            lf += [leaf, sp]; lt += [sp, leaf]
    d = W.graph_desc(8, 12, lf, lt, [50e9] * len(lf), [1e-6] * len(lf))
    rng = np.random.default_rng(1)
    src = rng.integers(0, 4, 2000).astype(np.int32)
    dst = rng.integers(4, 8, 2000).astype(np.int32)
    s = orc.Sim(d, 5)
    s.add_flows(src, dst, np.ones(2000), conn_id=np.arange(2000, dtype=np.int32) % 97)
    off, links = s.paths()
    lf, lt = np.array(lf), np.array(lt)
    via = np.zeros(2)
    seen = {}
    for f in range(2000):
        p = links[off[f]:off[f + 1]]
        assert len(p) == 4 and lf[p[0]] == src[f] and lt[p[-1]] == dst[f]
        assert all(lt[p[k]] == lf[p[k + 1]] for k in range(3))
        via[lt[p[1]] - 10] += 1
        key = (src[f], dst[f], f % 97)
        assert seen.setdefault(key, tuple(p)) == tuple(p)                 # same connection, same path
    assert abs(via[0] - via[1]) < 4 * np.sqrt(2000)
    s2 = orc.Sim(d, 6)
    s2.add_flows(src, dst, np.ones(2000), conn_id=np.arange(2000, dtype=np.int32) % 97)
    assert not np.array_equal(s2.paths()[1], links)                       # the seed moves flows
    # (4) a chain of 8 switches between two GPUs is too long; an isolated GPU is unreachable
    n = 10
    lf = [0] + list(range(2, n)) + [1]; lt = list(range(2, n)) + [1] + [0]
    s = orc.Sim(W.graph_desc(2, n, lf, lt, [1e9] * len(lf), [0.0] * len(lf)), 0)
    with pytest.raises(orc.OrcError):
        s.add_flows([0], [1], [1.0])
    s.add_flows([1], [0], [1e3])                                          # the way back is one link
    with pytest.raises(orc.OrcError):
        s.add_collective(orc.ALLGATHER_RING, [0, 1], 1e3)
    assert s.num_flows == 1


# ------------------------------------------------------------------------------------------------ S2 routing pins
def test_routing_leaf_spine_down_lane_comes_from_the_high_hash_word():
    """S2: with P parallel uplinks per (leaf, spine) the up lane is (H mod (n_spines P)) mod P and the down lane
    (H >> 32) mod P, H = mix(mix(mix(mix(seed) ^ src) ^ dst) ^ conn) with the published SplitMix64 step -- re-derived
    here in Python integers from the published constants, not from the oracle."""
    M = (1 << 64) - 1

    def mix(x):
        z = (x + 0x9E3779B97F4A7C15) & M
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
        return z ^ (z >> 31)

    assert mix(0) == 0xE220A8397B1DCDAF            # the published first output, so this restatement is pinned too
    P, nsp, G, seed = 4, 2, 32, 21
    d = W.topo_desc(W.TOPO_LEAF_SPINE, 8, 4, n_leaves=4, n_spines=nsp, uplinks_per_leaf_spine=P)
    rng = np.random.default_rng(2)
    src = rng.integers(0, G, 600).astype(np.int32)
    dst = ((src + rng.integers(1, G, 600)) % G).astype(np.int32)
    conn = rng.integers(0, 1000, 600).astype(np.int32)
    s = orc.Sim(d, seed)
    s.add_flows(src, dst, np.ones(600), conn_id=conn)
    off, links = s.paths()
    n_cross = 0
    for f in range(600):
        if src[f] // 8 == dst[f] // 8:             # same leaf (2 hosts x 4 GPUs per leaf)
            continue
        H = mix(mix(mix(mix(seed) ^ int(src[f])) ^ int(dst[f])) ^ int(conn[f]))
        c = H % (nsp * P)
        up = 4 * G + 2 * (((src[f] // 8) * nsp + c // P) * P + c % P)
        dn = 4 * G + 2 * (((dst[f] // 8) * nsp + c // P) * P + (H >> 32) % P) + 1
        assert list(links[off[f]:off[f + 1]]) == [2 * G + 2 * src[f], up, dn, 2 * G + 2 * dst[f] + 1]
        n_cross += 1
    assert n_cross > 300

def test_routing_structure_leaf_spine_and_balance():
    d = W.topo_desc(W.TOPO_LEAF_SPINE, 8, 4, n_leaves=4, n_spines=4, uplinks_per_leaf_spine=2)
    G, P, nsp = 32, 2, 4
    rng = np.random.default_rng(0)
    src = rng.integers(0, G, 4000).astype(np.int32)
    dst = (src + rng.integers(1, G, 4000)).astype(np.int32) % G
    s = orc.Sim(d, 7)
    s.add_flows(src, dst, np.ones(4000))
    off, links = s.paths()
    spine_hits = np.zeros(nsp * P)
    for f in range(4000):
        p = links[off[f]:off[f + 1]]
        hs, hd = src[f] // 4, dst[f] // 4
        if hs == hd:
            assert list(p) == [2 * src[f], 2 * dst[f] + 1]
        elif hs // 2 == hd // 2:
            assert list(p) == [2 * G + 2 * src[f], 2 * G + 2 * dst[f] + 1]
        else:
            assert len(p) == 4 and p[0] == 2 * G + 2 * src[f] and p[3] == 2 * G + 2 * dst[f] + 1
            u_up, u_dn = (p[1] - 4 * G) // 2, (p[2] - 4 * G) // 2
            assert (p[1] - 4 * G) % 2 == 0 and (p[2] - 4 * G) % 2 == 1
            assert u_up // (nsp * P) == hs // 2 and u_dn // (nsp * P) == hd // 2          # right leaves
            assert (u_up // P) % nsp == (u_dn // P) % nsp                                  # same spine
            spine_hits[u_up % (nsp * P)] += 1
    n = spine_hits.sum()
    chi2 = ((spine_hits - n / 8) ** 2 / (n / 8)).sum()
    assert chi2 < 30.0          # 7 dof; P(chi2 > 30) ~ 1e-4


def test_routing_fat_tree_structure_and_conn_persistence():
    k, U = 8, 2
    d = W.topo_desc(W.TOPO_FAT_TREE, k * k // 2, k // 2, k=k, agg_uplinks=U)
    G, h = k * k // 2 * (k // 2), k // 2
    s = orc.Sim(d, 3)
    # one ring over GPUs of different pods: every step of a pair reuses one path (conn = collective id)
    ranks = np.array([0, 17, 40, 100, 127], np.int32)
    s.add_collective(orc.ALLGATHER_RING, ranks, 1e6)
    off, links = s.paths()
    N = len(ranks)
    b1 = 4 * G
    b2 = b1 + 2 * k * h * h
    for f in range(s.num_flows):
        p = links[off[f]:off[f + 1]]
        assert list(p) == list(links[off[f % N]:off[f % N + 1]])
        a, b = ranks[f % N], ranks[(f + 1) % N]
        ha, hb = a // h, b // h
        assert len(p) == (4 if ha // h == hb // h else 6)
        if len(p) == 6:
            u1, u2, d2, d1 = (p[1] - b1) // 2, (p[2] - b2) // 2, (p[3] - b2) // 2, (p[4] - b1) // 2
            agg = u1 % h
            assert u1 // h == ha and d1 // h == hb and d1 % h == agg            # edge switches, same agg index
            assert u2 // U == (ha // h) * h + agg and d2 // U == (hb // h) * h + agg
            assert u2 % U == d2 % U                                              # same core
    # different seeds move some flows
    s2 = orc.Sim(d, 4)
    s2.add_collective(orc.ALLGATHER_RING, ranks, 1e6)
    assert not np.array_equal(s2.paths()[1], links)


# ------------------------------------------------------------------------------------------------ P9 invariances
def test_p9_byte_conservation_and_scaling():
    w = W.cfg4(batch=1, n_hosts=4, gph=4, n_leaves=2, n_spines=2)
    inst = w.instances[0]
    s = oracle_run(w.desc, inst, trace=True)
    ev, fl, rate, t0, t1 = s.trace()
    moved = np.zeros(s.num_flows)
    np.add.at(moved, fl, rate * (t1 - t0))
    np.testing.assert_allclose(moved, s.flows()[2], rtol=1e-9)
    # scale bytes and capacities by 2: times unchanged (up to the 2^-20 B/s rate grid)
    d2 = dict(w.desc, nvlink_Bps=2 * w.desc["nvlink_Bps"], nic_Bps=2 * w.desc["nic_Bps"],
              fabric_Bps=2 * w.desc["fabric_Bps"])
    op = inst.ops[0]
    inst2 = W.Instance(seed=inst.seed, ops=[W.RawFlows(op.src, op.dst, 2 * op.nbytes)])
    s2 = oracle_run(d2, inst2)
    np.testing.assert_allclose(s2.completion_times(), s.completion_times(), rtol=1e-12)
    assert np.array_equal(s2.bottlenecks(), s.bottlenecks())


def test_p9_locality_unrelated_traffic_does_not_change_a_single_bit():
    """Reading R-LZ (PAPER.md L128 / L167): a flow's state changes only when its own rate changes, so adding
    traffic that shares no link and no dependency with a set of flows leaves their completion times and
    bottlenecks BIT-identical, however many extra events it inserts into the clock."""
    d = single(n_hosts=2, gph=8)
    # group A: contended traffic among GPUs 0..3 and 8..11 (NVLink + NIC links of those GPUs only)
    src_a = [0, 1, 2, 3, 0, 1, 8, 9, 10, 0]
    dst_a = [8, 8, 8, 9, 1, 2, 0, 0, 1, 3]
    by_a = [3e6, 5e6, 7e6, 1.1e7, 2e6, 9e6, 4e6, 6e6, 1.3e7, 1e6]
    # group B: GPUs 4..7 and 12..15 only
    rng = np.random.default_rng(5)
    src_b = rng.integers(4, 8, 40); dst_b = rng.integers(12, 16, 40)
    by_b = np.floor(rng.uniform(1e5, 2e7, 40))
    a = run_flows(d, src_a, dst_a, by_a)
    ab = run_flows(d, list(src_a) + list(src_b), list(dst_a) + list(dst_b), list(by_a) + list(by_b))
    n = len(src_a)
    assert len(ab.event_log()) > len(a.event_log()) + 20           # B really interleaves its own events
    assert np.array_equal(ab.completion_times()[:n], a.completion_times())
    assert np.array_equal(ab.bottlenecks()[:n], a.bottlenecks())


def test_p9_history_partitions_every_flow_into_constant_rate_intervals():
    """Throughput history (PAPER.md L128 / L167): the recorded (time, rate) changes of a flow, closed by its
    completion time, add up to its size; rates within one interval set never exceed a link (checked at the sampled
    event times through the trace) and the first record of a flow is its activation."""
    w = W.cfg4(batch=1, n_hosts=4, gph=4, n_leaves=2, n_spines=2)
    o = oracle_run(w.desc, w.instances[0], trace=True)
    fl, t, r = o.history()
    td, (src, dst, nbytes, lat) = o.completion_times(), o.flows()
    assert np.array_equal(np.unique(fl), np.arange(o.num_flows))          # every flow has at least one record
    for f in range(o.num_flows):
        m = fl == f
        tt = np.append(t[m], td[f])
        assert np.all(np.diff(tt) >= 0) and np.all(r[m] > 0)
        assert tt[0] == lat[f]                                             # activation = start (0) + path latency
        assert abs(np.sum(r[m] * np.diff(tt)) - nbytes[f]) <= 1e-12 * nbytes[f]
    # the history is the trace with repeated rates dropped
    ev, tfl, trate, t0, t1 = o.trace()
    for f in (0, 7, 100):
        m = tfl == f
        rates, times = trate[m], t0[m]
        keep = np.append([True], rates[1:] != rates[:-1])
        assert np.array_equal(rates[keep], r[fl == f]) and np.array_equal(times[keep], t[fl == f])


def test_p9_run_until_is_a_prefix_of_the_full_run():
    """PAPER.md L167 "advancing the simulation ... up to a specified time": stopping at T changes nothing before T.
    Flows done by T have the times of the full run, the others are NaN / -1, and event log and throughput history
    are the full run's records with time <= T."""
    from util import oracle_build
    w = W.cfg1(batch=1, n_hosts=8, gph=4, n_leaves=4, n_spines=2)
    full = oracle_run(w.desc, w.instances[0])
    t_full, ev_full = full.completion_times(), full.event_log()
    ff, tf, rf = full.history()
    for T in (0.0, 0.25 * t_full.max(), 0.6 * t_full.max(), t_full.max(), 2 * t_full.max()):
        o = oracle_build(w.desc, w.instances[0])
        o.run(until=T)
        t = o.completion_times()
        done = t_full <= T
        assert np.array_equal(t[done], t_full[done]) and np.isnan(t[~done]).all()
        assert np.array_equal(o.bottlenecks()[done], full.bottlenecks()[done]) and np.all(o.bottlenecks()[~done] == -1)
        ev = o.event_log()
        assert np.array_equal(ev, ev_full[ev_full["t"] <= T])
        fo, to, ro = o.history()
        keep = tf <= T
        assert np.array_equal(fo, ff[keep]) and np.array_equal(to, tf[keep]) and np.array_equal(ro, rf[keep])
        ct, ct_full = o.collective_times(), full.collective_times()
        assert np.array_equal(ct[ct_full <= T], ct_full[ct_full <= T]) and np.isnan(ct[ct_full > T]).all()


def test_p9_single_spine_is_seed_independent():
    d = W.topo_desc(W.TOPO_LEAF_SPINE, 4, 4, n_leaves=2, n_spines=1, uplinks_per_leaf_spine=1)
    ops = [W.Coll(W.ALLREDUCE_RING, np.arange(0, 16, 2, dtype=np.int32), 32 * MiB),
           W.Coll(W.ALLTOALL, np.arange(16, dtype=np.int32), 8 * MiB, 1e-4)]
    a = oracle_run(d, W.Instance(seed=1, ops=ops))
    b = oracle_run(d, W.Instance(seed=99, ops=ops))
    assert np.array_equal(a.completion_times(), b.completion_times())
    assert np.array_equal(a.paths()[1], b.paths()[1])


# ------------------------------------------------------------------------------------------------ naive == fast
@pytest.mark.parametrize("wl", [
    lambda: W.cfg0(),
    lambda: W.cfg1(batch=2),
    lambda: W.cfg2(k=4, agg_uplinks=1),
    lambda: W.cfg3(batch=2),
    lambda: W.cfg4(batch=1, n_hosts=8, gph=4, n_leaves=4, n_spines=2),
])
def test_naive_and_fast_modes_bit_identical(wl):
    w = wl()
    inst = w.instances[-1]
    a = oracle_run(w.desc, inst, mode=orc.MODE_NAIVE)
    b = oracle_run(w.desc, inst, mode=orc.MODE_FAST)
    assert np.array_equal(a.completion_times(), b.completion_times())
    assert np.array_equal(a.bottlenecks(), b.bottlenecks())
    assert np.array_equal(a.event_log(), b.event_log())
    assert np.array_equal(completion_order(a.completion_times()), completion_order(b.completion_times()))
    assert not np.isnan(a.completion_times()).any()


# ------------------------------------------------------------------------------------------------ error behaviour
def test_input_validation():
    d = single()
    s = orc.Sim(d, 0)
    with pytest.raises(orc.OrcError):
        s.add_flows([0], [0], [1.0])                 # src == dst
    with pytest.raises(orc.OrcError):
        s.add_flows([0], [1], [0.0])                 # bytes <= 0
    with pytest.raises(orc.OrcError):
        s.add_flows([0], [99], [1.0])                # rank out of range
    with pytest.raises(orc.OrcError):
        s.add_collective(orc.ALLREDUCE_RING, [0, 1, 1], 1e6)   # duplicate rank
    with pytest.raises(orc.OrcError):
        s.add_flows([0], [1], [1.0], dep_off=[0, 1], dep_ids=[0])   # dep on itself / later flow
    assert s.num_flows == 0
    s.add_flows([0, 1], [1, 2], [1e6, 1e6], dep_off=[0, 0, 1], dep_ids=[0])
    s.run()
    t = s.completion_times()
    assert t[1] == pytest.approx(2 * (2e-6 + 1e6 / 450e9), rel=1e-12)
    s.add_flows([0], [1], [1.0])                     # after a run: a late submission (NEXT-1), not an error
    s.run()
    assert s.num_flows == 3 and not np.isnan(s.completion_times()).any()
