"""Shared test helpers: drive the CPU oracle from a neutral workload description."""
import numpy as np

from oracle import orc
from paper_2505_01616_b200 import workloads as W


def oracle_build(desc, inst, base_seed=0):
    """Oracle instance with the workload submitted but not run."""
    sim = orc.Sim(desc, seed=base_seed + inst.seed)
    cap = inst.capacities(desc, sim.num_links)
    if cap is not None:
        sim.set_link_capacities(cap)
    W.apply(inst,
            lambda kind, ranks, nbytes, start, after, chunks=1, after_flows=(): sim.add_collective(
                kind, ranks, nbytes, start, after, chunks, after_flows),
            lambda src, dst, nbytes, start, dep_off, dep_ids, conn: sim.add_flows(src, dst, nbytes, start, dep_off,
                                                                                   dep_ids, conn),
            lambda gpu, duration, lane, start, dep_off, dep_ids: sim.add_spans(gpu, duration, lane, start, dep_off,
                                                                               dep_ids))
    return sim


def oracle_run(desc, inst, mode=orc.MODE_NAIVE, trace=False, base_seed=0):
    sim = oracle_build(desc, inst, base_seed)
    sim.run(mode=mode, trace=trace)
    return sim


def completion_order(t_done):
    """O2: flows sorted by (t_done, flow id)."""
    return np.lexsort((np.arange(len(t_done)), t_done))
