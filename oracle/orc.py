"""ctypes wrapper of the CPU oracle (oracle/liborc.so).  TEST INFRASTRUCTURE ONLY.

Nothing here may be imported by the product package (paper_2505_01616_b200); only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs use it.
This module imports nothing from the product package either.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))

OK, EINVAL, ENOMEM, ECYCLE, ESTATE, ERANGE = 0, -1, -2, -4, -5, -6
TOPO_SINGLE, TOPO_LEAF_SPINE, TOPO_FAT_TREE, TOPO_GRAPH = 0, 1, 2, 3
ALLREDUCE_RING, ALLGATHER_RING, REDUCESCATTER_RING, ALLTOALL = 0, 1, 2, 3
BROADCAST_CHAIN, REDUCE_CHAIN, ALLREDUCE_TREE = 4, 5, 6
MODE_NAIVE, MODE_FAST = 0, 1
FLAG_SETTLE_EVERY_EVENT, FLAG_F64_SHARES = 1, 2     # orc_run_ex: SURVEY.md 8(c) S4.4 / S5 as written (see orc_netsim.h)


class TopologyDesc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n_hosts", C.c_int32), ("gpus_per_host", C.c_int32),
                ("nvlink_Bps", C.c_double), ("nic_Bps", C.c_double), ("fabric_Bps", C.c_double),
                ("hop_latency_s", C.c_double),
                ("n_leaves", C.c_int32), ("n_spines", C.c_int32), ("uplinks_per_leaf_spine", C.c_int32),
                ("k", C.c_int32), ("agg_uplinks", C.c_int32), ("compute_lanes", C.c_int32)]


EVENT_DTYPE = np.dtype([("t", "<f8"), ("n_completed", "<i4"), ("n_activated", "<i4"), ("n_rounds", "<i4"),
                        ("first_bneck", "<i4")])

_lib = None


def lib():
    global _lib
    if _lib is None:
        import importlib.util
        spec = importlib.util.spec_from_file_location("_orc_build", os.path.join(_HERE, "build_oracle.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        # ORC_LIB_PATH: a pre-built variant of the oracle (tests/test_oracle_mutants.py loads mutated copies through it)
        _lib = C.CDLL(os.environ.get("ORC_LIB_PATH") or mod.build())
        _lib.orc_mix64.restype = C.c_uint64
        _lib.orc_mix64.argtypes = [C.c_uint64]
        _lib.orc_destroy.restype = None
        _lib.orc_settle.restype = C.c_double
        _lib.orc_settle.argtypes = [C.c_double, C.c_double, C.c_double]
    return _lib


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


class OrcError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"{what}: oracle status {code}")
        self.code = code


def _chk(rc, what):
    if rc != OK:
        raise OrcError(rc, what)


def mix64(x: int) -> int:
    return int(lib().orc_mix64(C.c_uint64(x & 0xFFFFFFFFFFFFFFFF)))


def settle(rem, rate_Bps, dt):
    """S4.4 / Q11 settle step: max(rem - rate * dt, 0)."""
    return float(lib().orc_settle(rem, rate_Bps, dt))


def maxmin(cap, path_off, path, mode=MODE_NAIVE):
    """Stand-alone S5 solve.  Returns (rate[F], bneck[F], n_rounds, first_bneck)."""
    cap = np.ascontiguousarray(cap, dtype=np.float64)
    path_off = np.ascontiguousarray(path_off, dtype=np.int64)
    path = np.ascontiguousarray(path, dtype=np.int32)
    nf = len(path_off) - 1
    rate = np.zeros(nf, dtype=np.float64)
    bneck = np.zeros(nf, dtype=np.int32)
    R, fb = C.c_int32(0), C.c_int32(0)
    _chk(lib().orc_maxmin(C.c_int32(len(cap)), _p(cap, C.c_double), C.c_int32(nf), _p(path_off, C.c_int64),
                          _p(path, C.c_int32), C.c_int32(mode), _p(rate, C.c_double), _p(bneck, C.c_int32),
                          C.byref(R), C.byref(fb)), "orc_maxmin")
    return rate, bneck, R.value, fb.value


class Sim:
    """One oracle simulation instance (the oracle has no batch dimension)."""

    def __init__(self, desc: dict, seed: int = 0):
        self._h = C.c_void_p()
        if "graph" in desc:          # user-supplied topology (NEXT-4): link list between nodes, GPUs are nodes 0..G-1
            g = desc["graph"]
            lf = np.ascontiguousarray(g["link_from"], dtype=np.int32); lt = np.ascontiguousarray(g["link_to"], dtype=np.int32)
            cap = np.ascontiguousarray(g["cap_Bps"], dtype=np.float64); lat = np.ascontiguousarray(g["latency_s"], dtype=np.float64)
            _chk(lib().orc_create_topology_graph(C.c_int32(g["n_gpus"]), C.c_int32(g["n_nodes"]), C.c_int32(len(lf)),
                                                 _p(lf, C.c_int32), _p(lt, C.c_int32), _p(cap, C.c_double),
                                                 _p(lat, C.c_double), C.c_int32(g.get("compute_lanes", 0)),
                                                 C.c_uint64(seed), C.byref(self._h)), "orc_create_topology_graph")
            return
        d = TopologyDesc(**desc)
        _chk(lib().orc_create_topology(C.byref(d), C.c_uint64(seed), C.byref(self._h)), "orc_create_topology")

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def num_links(self):
        n = C.c_int32()
        _chk(lib().orc_num_links(self._h, C.byref(n)), "orc_num_links")
        return n.value

    def set_link_capacities(self, cap):
        cap = np.ascontiguousarray(cap, dtype=np.float64)
        assert len(cap) == self.num_links
        _chk(lib().orc_set_link_capacities(self._h, _p(cap, C.c_double)), "orc_set_link_capacities")

    def link_capacities(self):
        cap = np.zeros(self.num_links, dtype=np.float64)
        _chk(lib().orc_get_link_capacities(self._h, _p(cap, C.c_double)), "orc_get_link_capacities")
        return cap

    def add_collective(self, kind, ranks, nbytes, start=0.0, after=(), chunks=1, after_flows=()):
        ranks = np.ascontiguousarray(ranks, dtype=np.int32)
        after = np.ascontiguousarray(after, dtype=np.int32)
        after_flows = np.ascontiguousarray(after_flows, dtype=np.int64)
        cid = C.c_int32()
        _chk(lib().orc_add_collective_full(self._h, C.c_int32(kind), _p(ranks, C.c_int32), C.c_int32(len(ranks)),
                                           C.c_double(nbytes), C.c_double(start),
                                           _p(after, C.c_int32) if len(after) else None, C.c_int32(len(after)),
                                           _p(after_flows, C.c_int64) if len(after_flows) else None,
                                           C.c_int32(len(after_flows)), C.c_int32(chunks), C.byref(cid)),
             "orc_add_collective_full")
        return cid.value

    def add_spans(self, gpu, duration, lane=None, start=None, dep_off=None, dep_ids=None):
        gpu = np.ascontiguousarray(gpu, dtype=np.int32)
        duration = np.ascontiguousarray(duration, dtype=np.float64)
        lane = None if lane is None else np.ascontiguousarray(lane, dtype=np.int32)
        start = None if start is None else np.ascontiguousarray(start, dtype=np.float64)
        dep_off = None if dep_off is None else np.ascontiguousarray(dep_off, dtype=np.int64)
        dep_ids = None if dep_ids is None else np.ascontiguousarray(dep_ids, dtype=np.int64)
        first = C.c_int64()
        _chk(lib().orc_add_spans(self._h, C.c_int64(len(gpu)), _p(gpu, C.c_int32), _p(lane, C.c_int32),
                                 _p(duration, C.c_double), _p(start, C.c_double), _p(dep_off, C.c_int64),
                                 _p(dep_ids, C.c_int64), C.byref(first)), "orc_add_spans")
        return first.value

    def add_flows(self, src, dst, nbytes, start=None, dep_off=None, dep_ids=None, conn_id=None):
        src = np.ascontiguousarray(src, dtype=np.int32)
        dst = np.ascontiguousarray(dst, dtype=np.int32)
        nbytes = np.ascontiguousarray(nbytes, dtype=np.float64)
        start = None if start is None else np.ascontiguousarray(start, dtype=np.float64)
        dep_off = None if dep_off is None else np.ascontiguousarray(dep_off, dtype=np.int64)
        dep_ids = None if dep_ids is None else np.ascontiguousarray(dep_ids, dtype=np.int64)
        conn_id = None if conn_id is None else np.ascontiguousarray(conn_id, dtype=np.int32)
        first = C.c_int64()
        _chk(lib().orc_add_flows(self._h, C.c_int64(len(src)), _p(src, C.c_int32), _p(dst, C.c_int32),
                                 _p(nbytes, C.c_double), _p(start, C.c_double), _p(dep_off, C.c_int64),
                                 _p(dep_ids, C.c_int64), _p(conn_id, C.c_int32), C.byref(first)), "orc_add_flows")
        return first.value

    def run(self, mode=MODE_NAIVE, trace=False, until=None, flags=0):
        if flags:
            _chk(lib().orc_run_ex(self._h, C.c_int32(mode), C.c_int32(1 if trace else 0),
                                  C.c_double(float("inf") if until is None else until), C.c_int32(flags)), "orc_run_ex")
        elif until is None:
            _chk(lib().orc_run(self._h, C.c_int32(mode), C.c_int32(1 if trace else 0)), "orc_run")
        else:
            _chk(lib().orc_run_until(self._h, C.c_int32(mode), C.c_int32(1 if trace else 0), C.c_double(until)),
                 "orc_run_until")

    def rollback(self, T):
        _chk(lib().orc_rollback(self._h, C.c_double(T)), "orc_rollback")

    def update_flow_start(self, flow, start):
        _chk(lib().orc_update_flow_start(self._h, C.c_int64(flow), C.c_double(start)), "orc_update_flow_start")

    def gc(self, T):
        _chk(lib().orc_gc(self._h, C.c_double(T)), "orc_gc")

    @property
    def num_flows(self):
        n = C.c_int64()
        _chk(lib().orc_num_flows(self._h, C.byref(n)), "orc_num_flows")
        return n.value

    @property
    def num_collectives(self):
        n = C.c_int32()
        _chk(lib().orc_num_collectives(self._h, C.byref(n)), "orc_num_collectives")
        return n.value

    def completion_times(self):
        out = np.zeros(self.num_flows, dtype=np.float64)
        _chk(lib().orc_get_completion_times(self._h, _p(out, C.c_double), C.c_int64(len(out))), "orc_get_completion_times")
        return out

    def bottlenecks(self):
        out = np.zeros(self.num_flows, dtype=np.int32)
        _chk(lib().orc_get_bottlenecks(self._h, _p(out, C.c_int32), C.c_int64(len(out))), "orc_get_bottlenecks")
        return out

    def collective_times(self):
        out = np.zeros(self.num_collectives, dtype=np.float64)
        _chk(lib().orc_get_collective_times(self._h, _p(out, C.c_double), C.c_int32(len(out))), "orc_get_collective_times")
        return out

    def event_log(self):
        n = C.c_int64()
        _chk(lib().orc_num_events(self._h, C.byref(n)), "orc_num_events")
        out = np.zeros(n.value, dtype=EVENT_DTYPE)
        _chk(lib().orc_get_event_log(self._h, C.c_void_p(out.ctypes.data), C.c_int64(n.value), C.byref(n)),
             "orc_get_event_log")
        return out

    def paths(self):
        n = C.c_int64()
        _chk(lib().orc_num_path_entries(self._h, C.byref(n)), "orc_num_path_entries")
        off = np.zeros(self.num_flows + 1, dtype=np.int64)
        links = np.zeros(n.value, dtype=np.int32)
        _chk(lib().orc_get_paths(self._h, _p(off, C.c_int64), _p(links, C.c_int32), C.c_int64(n.value)), "orc_get_paths")
        return off, links

    def flows(self):
        F = self.num_flows
        src = np.zeros(F, np.int32); dst = np.zeros(F, np.int32)
        b = np.zeros(F, np.float64); lat = np.zeros(F, np.float64)
        _chk(lib().orc_get_flow_endpoints(self._h, _p(src, C.c_int32), _p(dst, C.c_int32), _p(b, C.c_double),
                                          _p(lat, C.c_double), C.c_int64(F)), "orc_get_flow_endpoints")
        return src, dst, b, lat

    def preds(self):
        n = C.c_int64()
        _chk(lib().orc_get_preds(self._h, None, None, C.c_int64(0), C.byref(n)), "orc_get_preds")
        off = np.zeros(self.num_flows + 1, dtype=np.int64)
        pr = np.zeros(n.value, dtype=np.int32)
        _chk(lib().orc_get_preds(self._h, _p(off, C.c_int64), _p(pr, C.c_int32), C.c_int64(n.value), C.byref(n)),
             "orc_get_preds")
        return off, pr

    def work_counters(self):
        out = np.zeros(7, dtype=np.float64)
        _chk(lib().orc_get_work_counters(self._h, _p(out, C.c_double)), "orc_get_work_counters")
        return dict(zip(["sum_A", "sum_Ah", "sum_R", "sum_LamR", "sum_Lam", "completions", "events"], out.tolist()))

    def history(self):
        """Throughput history: (flow, t, rate) per rate change, sorted by (flow, t)."""
        n = C.c_int64()
        _chk(lib().orc_history_size(self._h, C.byref(n)), "orc_history_size")
        fl = np.zeros(n.value, np.int32); t = np.zeros(n.value, np.float64); rate = np.zeros(n.value, np.float64)
        _chk(lib().orc_get_history(self._h, _p(fl, C.c_int32), _p(t, C.c_double), _p(rate, C.c_double),
                                   C.c_int64(n.value)), "orc_get_history")
        order = np.lexsort((t, fl))
        return fl[order], t[order], rate[order]

    def trace(self):
        n = C.c_int64()
        _chk(lib().orc_trace_size(self._h, C.byref(n)), "orc_trace_size")
        ev = np.zeros(n.value, np.int64); fl = np.zeros(n.value, np.int32)
        rate = np.zeros(n.value, np.float64); t0 = np.zeros(n.value, np.float64); t1 = np.zeros(n.value, np.float64)
        _chk(lib().orc_get_trace(self._h, _p(ev, C.c_int64), _p(fl, C.c_int32), _p(rate, C.c_double),
                                 _p(t0, C.c_double), _p(t1, C.c_double), C.c_int64(n.value)), "orc_get_trace")
        return ev, fl, rate, t0, t1
