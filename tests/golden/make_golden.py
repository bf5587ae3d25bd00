"""Writes the stored expected values for the full-size parity cases: cfg2 (its one instance) and cfg4 (all eight
instances of the batch bench.py times).

Calls ONLY the CPU oracle (oracle/, fast mode) on the seeded inputs of paper_2505_01616_b200/workloads.py; nothing
here touches the CUDA path.  One instance takes ~5 min (cfg4) or ~12 min (cfg2) of one CPU core; the instances
of cfg4 run as separate processes.

    python tests/golden/make_golden.py [cfg4] [cfg2] [a2a304] [cfg4:3]        # cfg4:3 = only instance 3 of cfg4

Per instance the file holds: 4096 sampled flows (index, completion time, bottleneck), the SHA-256 of ALL completion
times, of ALL bottleneck ids and of the `t` column of the event log, the event count, the oracle's work counters
(the roofline's algorithmic bytes) and the wall time of the run.
"""
import hashlib
import os
import subprocess
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

from oracle import orc  # noqa: E402
from paper_2505_01616_b200 import workloads as W  # noqa: E402
from util import oracle_run  # noqa: E402

CFG4_BATCH = 8


def a2a304():
    """A unit that fits no 16-CTA cluster (grid path): cfg4's recipe on 304 GPUs = 92,112 concurrent flows."""
    return W.cfg4(batch=1, n_hosts=38, gph=8, n_leaves=2, n_spines=4)


def make(name, inst):
    w = W.cfg4(batch=CFG4_BATCH) if name == "cfg4" else a2a304() if name == "a2a304" else W.cfg2()
    t0 = time.time()
    o = oracle_run(w.desc, w.instances[inst], mode=orc.MODE_FAST, base_seed=w.base_seed)
    t = o.completion_times()
    b = o.bottlenecks()
    ev = o.event_log()
    rng = np.random.default_rng(12345 + inst)
    idx = np.sort(rng.choice(len(t), size=4096, replace=False))
    wk = o.work_counters()   # per-event work summed over the run (the roofline's algorithmic bytes)
    secs = time.time() - t0
    np.savez_compressed(os.path.join(HERE, f"{name}_inst{inst}.npz"), idx=idx, t_done=t[idx], bneck=b[idx],
                        n_events=np.int64(len(ev)), sha_t=np.array(hashlib.sha256(t.tobytes()).hexdigest()),
                        sha_bneck=np.array(hashlib.sha256(b.tobytes()).hexdigest()),
                        sha_event_t=np.array(hashlib.sha256(np.ascontiguousarray(ev["t"]).tobytes()).hexdigest()),
                        work_keys=np.array(sorted(wk)), work_vals=np.array([wk[k] for k in sorted(wk)], np.float64),
                        oracle_seconds=np.float64(secs), n_flows=np.int64(len(t)))
    print(name, "instance", inst, "flows", len(t), "events", len(ev), "oracle seconds", round(secs, 1), flush=True)


if __name__ == "__main__":
    jobs = []
    for a in (sys.argv[1:] or ["cfg4", "cfg2"]):
        if ":" in a:
            n, i = a.split(":")
            make(n, int(i))
        elif a == "cfg4":       # one process per instance
            jobs += [subprocess.Popen([sys.executable, os.path.abspath(__file__), f"cfg4:{i}"]) for i in range(CFG4_BATCH)]
        else:
            make(a, 0)
    for j in jobs:
        if j.wait() != 0:
            raise SystemExit("a golden job failed")
