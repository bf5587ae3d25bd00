"""Writes the stored expected values for the full-size parity cases (cfg2, cfg4 instance 0).

Calls ONLY the CPU oracle (oracle/, fast mode) on the seeded inputs of paper_2505_01616_b200/workloads.py; nothing
here touches the CUDA path.  Takes ~4 min (cfg4) and ~12 min (cfg2) of one CPU core.

    python tests/golden/make_golden.py [cfg4] [cfg2]
"""
import hashlib
import os
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


def make(name):
    w = W.cfg4(batch=1) if name == "cfg4" else W.cfg2()
    t0 = time.time()
    o = oracle_run(w.desc, w.instances[0], mode=orc.MODE_FAST, base_seed=w.base_seed)
    t = o.completion_times()
    b = o.bottlenecks()
    rng = np.random.default_rng(12345)
    idx = np.sort(rng.choice(len(t), size=4096, replace=False))
    wk = o.work_counters()   # per-event work summed over the run (the roofline's algorithmic bytes)
    secs = time.time() - t0
    np.savez_compressed(os.path.join(HERE, f"{name}_inst0.npz"), idx=idx, t_done=t[idx], bneck=b[idx],
                        n_events=np.int64(len(o.event_log())), sha_t=np.array(hashlib.sha256(t.tobytes()).hexdigest()),
                        work_keys=np.array(sorted(wk)), work_vals=np.array([wk[k] for k in sorted(wk)], np.float64),
                        oracle_seconds=np.float64(secs), n_flows=np.int64(len(t)))
    print(name, "flows", len(t), "events", len(o.event_log()), "oracle seconds", round(time.time() - t0, 1))


if __name__ == "__main__":
    for n in (sys.argv[1:] or ["cfg4", "cfg2"]):
        make(n)
