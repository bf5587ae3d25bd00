"""Thin ctypes binding of libphs.so (include/phs.h).  Argument marshalling only: every step of the hot path runs
in the library's CUDA kernels.  There is no CPU fallback -- if the library is missing or no CUDA device is usable
the calls raise.

The module-level functions carry the C names (phs_create_topology, phs_add_collective, phs_add_flows, phs_run,
phs_get_completion_times, ...); `Sim` is a small convenience wrapper around a handle.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libphs.so")

PHS_OK, PHS_EINVAL, PHS_ENOMEM, PHS_ECUDA, PHS_ECYCLE, PHS_ESTATE, PHS_ERANGE = 0, -1, -2, -3, -4, -5, -6
TOPO_SINGLE, TOPO_LEAF_SPINE, TOPO_FAT_TREE = 0, 1, 2
ALLREDUCE_RING, ALLGATHER_RING, REDUCESCATTER_RING, ALLTOALL = 0, 1, 2, 3
BROADCAST_CHAIN, REDUCE_CHAIN, ALLREDUCE_TREE = 4, 5, 6


class TopologyDesc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n_hosts", C.c_int32), ("gpus_per_host", C.c_int32),
                ("nvlink_Bps", C.c_double), ("nic_Bps", C.c_double), ("fabric_Bps", C.c_double),
                ("hop_latency_s", C.c_double),
                ("n_leaves", C.c_int32), ("n_spines", C.c_int32), ("uplinks_per_leaf_spine", C.c_int32),
                ("k", C.c_int32), ("agg_uplinks", C.c_int32), ("compute_lanes", C.c_int32)]


class Counters(C.Structure):
    _fields_ = [("n_events", C.c_int64), ("n_flow_events", C.c_int64), ("sum_active", C.c_int64),
                ("sum_par_rounds", C.c_int64), ("n_kernel_launches", C.c_int64), ("h2d_bytes", C.c_int64),
                ("max_active", C.c_int32), ("max_slots", C.c_int32), ("cluster_size", C.c_int32),
                ("clusters_resident", C.c_int32), ("resumed_units", C.c_int32), ("window_gang", C.c_int32),
                ("main_kernel_ms", C.c_double), ("grid_ctas", C.c_int32), ("pad_", C.c_int32), ("resumed_from_s", C.c_double), ("n_windows", C.c_int64)]


EVENT_DTYPE = np.dtype([("t", "<f8"), ("n_completed", "<i4"), ("n_activated", "<i4"), ("n_rounds", "<i4"),
                        ("first_bneck", "<i4")])

# every symbol include/phs.h declares (tests check that the library exports all of them)
SYMBOLS = ["phs_create_topology", "phs_create_topology_graph", "phs_destroy", "phs_num_links", "phs_batch", "phs_set_link_capacities",
           "phs_set_link_capacities_batch",
           "phs_get_link_capacities", "phs_add_collective", "phs_add_collective_ex", "phs_add_collective_full", "phs_add_spans", "phs_add_collective_batch", "phs_add_flows",
           "phs_enable_event_log", "phs_enable_history", "phs_get_flow_history", "phs_set_scheduler",
           "phs_set_decomposition", "phs_set_devices", "phs_instance_device", "phs_set_windows", "phs_set_snapshots", "phs_update_flow_start", "phs_rollback", "phs_gc",
           "phs_finalize", "phs_run", "phs_run_until", "phs_run_static", "phs_num_flows", "phs_total_flows",
           "phs_num_collectives", "phs_get_completion_times", "phs_get_bottlenecks",
           "phs_get_all_completion_times", "phs_get_all_bottlenecks", "phs_get_collective_times",
           "phs_get_event_log", "phs_num_path_entries", "phs_get_paths", "phs_get_link_flows", "phs_get_preds", "phs_get_flow_table",
           "phs_get_counters", "phs_instance_path", "phs_last_error"]

_lib = None


class PhsError(RuntimeError):
    def __init__(self, code, what, msg):
        super().__init__(f"{what} failed with status {code}: {msg}")
        self.code = code


def lib():
    """Loads libphs.so (building nothing: use `python -m paper_2505_01616_b200.build`).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2505_01616_b200.build` "
                              "(there is no CPU fallback)")
        _lib = C.CDLL(_LIB_PATH)
        _lib.phs_last_error.restype = C.c_char_p
        _lib.phs_instance_path.restype = C.c_char_p
        _lib.phs_instance_path.argtypes = [C.c_void_p, C.c_int32]
        _lib.phs_destroy.restype = None
        _lib.phs_destroy.argtypes = [C.c_void_p]
    return _lib


def _chk(rc, what):
    if rc != PHS_OK:
        raise PhsError(rc, what, lib().phs_last_error().decode())


def _arr(a, dt):
    return None if a is None else np.ascontiguousarray(a, dtype=dt)


def _p(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


# ---------------------------------------------------------------------------------------------- C-named calls
def phs_create_topology(desc: dict, seed: int, batch: int):
    h = C.c_void_p()
    if "graph" in desc:          # user-supplied topology: workloads.graph_desc
        g = desc["graph"]
        lf, lt = _arr(g["link_from"], np.int32), _arr(g["link_to"], np.int32)
        cap, lat = _arr(g["cap_Bps"], np.float64), _arr(g["latency_s"], np.float64)
        if not (len(lf) == len(lt) == len(cap) == len(lat)):
            raise ValueError("link arrays have inconsistent lengths")
        _chk(lib().phs_create_topology_graph(C.c_int32(g["n_gpus"]), C.c_int32(g["n_nodes"]), C.c_int32(len(lf)), _p(lf),
                                             _p(lt), _p(cap), _p(lat), C.c_int32(g.get("compute_lanes", 0)),
                                             C.c_uint64(seed), C.c_int32(batch), C.byref(h)), "phs_create_topology_graph")
        return h
    d = TopologyDesc(**desc)
    _chk(lib().phs_create_topology(C.byref(d), C.c_uint64(seed), C.c_int32(batch), C.byref(h)), "phs_create_topology")
    return h


def phs_destroy(h):
    lib().phs_destroy(h)


def phs_num_links(h):
    n = C.c_int32()
    _chk(lib().phs_num_links(h, C.byref(n)), "phs_num_links")
    return n.value


def phs_set_link_capacities(h, instance, cap):
    cap = _arr(cap, np.float64)
    if len(cap) != phs_num_links(h):
        raise ValueError("capacity array must have n_links entries")
    _chk(lib().phs_set_link_capacities(h, C.c_int32(instance), _p(cap)), "phs_set_link_capacities")


def phs_set_link_capacities_batch(h, cap):
    cap = _arr(cap, np.float64)
    b = C.c_int32()
    _chk(lib().phs_batch(h, C.byref(b)), "phs_batch")
    if cap.shape != (b.value, phs_num_links(h)):
        raise ValueError("capacity array must be [batch][n_links]")
    _chk(lib().phs_set_link_capacities_batch(h, _p(cap)), "phs_set_link_capacities_batch")


def phs_get_link_capacities(h, instance):
    cap = np.zeros(phs_num_links(h), np.float64)
    _chk(lib().phs_get_link_capacities(h, C.c_int32(instance), _p(cap)), "phs_get_link_capacities")
    return cap


def phs_add_collective(h, instance, kind, ranks, nbytes, start=0.0, after=(), chunks=1, after_flows=()):
    ranks = _arr(ranks, np.int32)
    after = _arr(after, np.int32)
    after_flows = _arr(after_flows, np.int64)
    cid = C.c_int32()
    if chunks == 1 and not len(after_flows):
        _chk(lib().phs_add_collective(h, C.c_int32(instance), C.c_int32(kind), _p(ranks), C.c_int32(len(ranks)),
                                      C.c_double(nbytes), C.c_double(start), _p(after) if len(after) else None,
                                      C.c_int32(len(after)), C.byref(cid)), "phs_add_collective")
    else:
        _chk(lib().phs_add_collective_full(h, C.c_int32(instance), C.c_int32(kind), _p(ranks), C.c_int32(len(ranks)),
                                           C.c_double(nbytes), C.c_double(start), _p(after) if len(after) else None,
                                           C.c_int32(len(after)), _p(after_flows) if len(after_flows) else None,
                                           C.c_int32(len(after_flows)), C.c_int32(chunks), C.byref(cid)),
             "phs_add_collective_full")
    return cid.value


def phs_add_spans(h, instance, gpu, duration, lane=None, start=None, dep_off=None, dep_ids=None):
    gpu, lane = _arr(gpu, np.int32), _arr(lane, np.int32)
    duration, start = _arr(duration, np.float64), _arr(start, np.float64)
    dep_off, dep_ids = _arr(dep_off, np.int64), _arr(dep_ids, np.int64)
    n = len(gpu)
    if len(duration) != n or (lane is not None and len(lane) != n) or (start is not None and len(start) != n) or \
            (dep_off is not None and len(dep_off) != n + 1):
        raise ValueError("span arrays have inconsistent lengths")
    first = C.c_int64()
    _chk(lib().phs_add_spans(h, C.c_int32(instance), C.c_int64(n), _p(gpu), _p(lane), _p(duration), _p(start),
                             _p(dep_off), _p(dep_ids), C.byref(first)), "phs_add_spans")
    return first.value


def phs_add_collective_batch(h, kind, ranks, nbytes, start=None, after=()):
    ranks = _arr(ranks, np.int32)
    after = _arr(after, np.int32)
    nbytes = _arr(nbytes, np.float64)
    start = _arr(start, np.float64)
    b = C.c_int32()
    _chk(lib().phs_batch(h, C.byref(b)), "phs_batch")
    if len(nbytes) != b.value or (start is not None and len(start) != b.value):
        raise ValueError("per-instance arrays must have `batch` entries")
    cid = C.c_int32()
    _chk(lib().phs_add_collective_batch(h, C.c_int32(kind), _p(ranks), C.c_int32(len(ranks)), _p(nbytes), _p(start),
                                        _p(after) if len(after) else None, C.c_int32(len(after)), C.byref(cid)),
         "phs_add_collective_batch")
    return cid.value


def phs_add_flows(h, instance, src, dst, nbytes, start=None, dep_off=None, dep_ids=None, conn_id=None):
    src, dst = _arr(src, np.int32), _arr(dst, np.int32)
    nbytes, start = _arr(nbytes, np.float64), _arr(start, np.float64)
    dep_off, dep_ids, conn_id = _arr(dep_off, np.int64), _arr(dep_ids, np.int64), _arr(conn_id, np.int32)
    n = len(src)
    if len(dst) != n or len(nbytes) != n or (start is not None and len(start) != n) or \
            (dep_off is not None and len(dep_off) != n + 1) or (conn_id is not None and len(conn_id) != n):
        raise ValueError("flow arrays have inconsistent lengths")
    first = C.c_int64()
    _chk(lib().phs_add_flows(h, C.c_int32(instance), C.c_int64(n), _p(src), _p(dst), _p(nbytes), _p(start),
                             _p(dep_off), _p(dep_ids), _p(conn_id), C.byref(first)), "phs_add_flows")
    return first.value


def phs_enable_event_log(h, enable=True):
    _chk(lib().phs_enable_event_log(h, C.c_int32(1 if enable else 0)), "phs_enable_event_log")


def phs_set_scheduler(h, path=0, cta_slots=0):
    _chk(lib().phs_set_scheduler(h, C.c_int32(path), C.c_int32(cta_slots)), "phs_set_scheduler")


def phs_enable_history(h, max_records):
    _chk(lib().phs_enable_history(h, C.c_int64(max_records)), "phs_enable_history")


def phs_get_flow_history(h, instance):
    """(off[F+1], t[n], rate_Bps[n]): the rate changes of every flow of the instance, chronological per flow."""
    n = C.c_int64()
    _chk(lib().phs_get_flow_history(h, C.c_int32(instance), None, None, None, C.c_int64(0), C.byref(n)),
         "phs_get_flow_history")
    F = phs_num_flows(h, instance)
    off = np.zeros(F + 1, np.int64); t = np.zeros(n.value, np.float64); rate = np.zeros(n.value, np.float64)
    _chk(lib().phs_get_flow_history(h, C.c_int32(instance), _p(off), _p(t), _p(rate), C.c_int64(n.value),
                                    C.byref(n)), "phs_get_flow_history")
    return off, t, rate


def phs_set_decomposition(h, enable=True):
    _chk(lib().phs_set_decomposition(h, C.c_int32(1 if enable else 0)), "phs_set_decomposition")


def phs_set_windows(h, enable=True):
    _chk(lib().phs_set_windows(h, C.c_int32(1 if enable else 0)), "phs_set_windows")


def phs_set_devices(h, device_ids):
    d = _arr(device_ids, np.int32)
    _chk(lib().phs_set_devices(h, C.c_int32(len(d)), _p(d)), "phs_set_devices")


def phs_instance_device(h, instance):
    d = C.c_int32()
    _chk(lib().phs_instance_device(h, C.c_int32(instance), C.byref(d)), "phs_instance_device")
    return d.value


def phs_set_snapshots(h, n):
    _chk(lib().phs_set_snapshots(h, C.c_int32(n)), "phs_set_snapshots")


def phs_update_flow_start(h, instance, flow, start):
    _chk(lib().phs_update_flow_start(h, C.c_int32(instance), C.c_int64(flow), C.c_double(start)), "phs_update_flow_start")


def phs_rollback(h, t):
    _chk(lib().phs_rollback(h, C.c_double(t)), "phs_rollback")


def phs_gc(h, t):
    _chk(lib().phs_gc(h, C.c_double(t)), "phs_gc")


def phs_finalize(h, stream=None):
    _chk(lib().phs_finalize(h, C.c_void_p(stream or 0)), "phs_finalize")


def phs_run_until(h, t_stop_s, stream=None):
    _chk(lib().phs_run_until(h, C.c_double(t_stop_s), C.c_void_p(stream or 0)), "phs_run_until")


def phs_run(h, stream=None):
    _chk(lib().phs_run(h, C.c_void_p(stream or 0)), "phs_run")


PHS_STATIC_SCRATCH_BYTES = 8 << 20
PHS_STATIC_MAX_UNITS = 4096


def phs_run_static(h, t_done_dev, bneck_dev, n, stream=None):
    """t_done_dev / bneck_dev: DEVICE addresses (int, e.g. torch.Tensor.data_ptr()) of n doubles / n int32, or None."""
    _chk(lib().phs_run_static(h, C.c_void_p(stream or 0), C.c_void_p(t_done_dev or 0), C.c_void_p(bneck_dev or 0),
                              C.c_int64(n)), "phs_run_static")


def phs_num_flows(h, instance):
    n = C.c_int64()
    _chk(lib().phs_num_flows(h, C.c_int32(instance), C.byref(n)), "phs_num_flows")
    return n.value


def phs_total_flows(h):
    n = C.c_int64()
    _chk(lib().phs_total_flows(h, C.byref(n)), "phs_total_flows")
    return n.value


def phs_num_collectives(h, instance):
    n = C.c_int32()
    _chk(lib().phs_num_collectives(h, C.c_int32(instance), C.byref(n)), "phs_num_collectives")
    return n.value


def phs_get_completion_times(h, instance, out=None, device_ptr=None):
    """Host numpy array by default; with device_ptr (int, e.g. torch.Tensor.data_ptr()) fills device memory."""
    n = phs_num_flows(h, instance)
    if device_ptr is not None:
        _chk(lib().phs_get_completion_times(h, C.c_int32(instance), C.c_void_p(device_ptr), C.c_int64(n), C.c_int32(1)),
             "phs_get_completion_times")
        return None
    out = np.empty(n, np.float64) if out is None else out
    _chk(lib().phs_get_completion_times(h, C.c_int32(instance), _p(out), C.c_int64(n), C.c_int32(0)),
         "phs_get_completion_times")
    return out


def phs_get_bottlenecks(h, instance, out=None, device_ptr=None):
    n = phs_num_flows(h, instance)
    if device_ptr is not None:
        _chk(lib().phs_get_bottlenecks(h, C.c_int32(instance), C.c_void_p(device_ptr), C.c_int64(n), C.c_int32(1)),
             "phs_get_bottlenecks")
        return None
    out = np.empty(n, np.int32) if out is None else out
    _chk(lib().phs_get_bottlenecks(h, C.c_int32(instance), _p(out), C.c_int64(n), C.c_int32(0)), "phs_get_bottlenecks")
    return out


def phs_get_all_completion_times(h, out=None, device_ptr=None):
    n = phs_total_flows(h)
    if device_ptr is not None:
        _chk(lib().phs_get_all_completion_times(h, C.c_void_p(device_ptr), C.c_int64(n), C.c_int32(1)),
             "phs_get_all_completion_times")
        return None
    out = np.empty(n, np.float64) if out is None else out
    _chk(lib().phs_get_all_completion_times(h, _p(out), C.c_int64(n), C.c_int32(0)), "phs_get_all_completion_times")
    return out


def phs_get_all_bottlenecks(h, out=None, device_ptr=None):
    n = phs_total_flows(h)
    if device_ptr is not None:
        _chk(lib().phs_get_all_bottlenecks(h, C.c_void_p(device_ptr), C.c_int64(n), C.c_int32(1)),
             "phs_get_all_bottlenecks")
        return None
    out = np.empty(n, np.int32) if out is None else out
    _chk(lib().phs_get_all_bottlenecks(h, _p(out), C.c_int64(n), C.c_int32(0)), "phs_get_all_bottlenecks")
    return out


def phs_get_collective_times(h, instance):
    n = phs_num_collectives(h, instance)
    out = np.empty(n, np.float64)
    _chk(lib().phs_get_collective_times(h, C.c_int32(instance), _p(out), C.c_int32(n)), "phs_get_collective_times")
    return out


def phs_get_event_log(h, instance):
    n = C.c_int64()
    _chk(lib().phs_get_event_log(h, C.c_int32(instance), None, C.c_int64(0), C.byref(n)), "phs_get_event_log")
    out = np.zeros(n.value, EVENT_DTYPE)
    _chk(lib().phs_get_event_log(h, C.c_int32(instance), _p(out), C.c_int64(n.value), C.byref(n)), "phs_get_event_log")
    return out


def phs_get_paths(h, instance):
    n = C.c_int64()
    _chk(lib().phs_num_path_entries(h, C.c_int32(instance), C.byref(n)), "phs_num_path_entries")
    off = np.zeros(phs_num_flows(h, instance) + 1, np.int64)
    links = np.zeros(n.value, np.int32)
    _chk(lib().phs_get_paths(h, C.c_int32(instance), _p(off), _p(links), C.c_int64(n.value)), "phs_get_paths")
    return off, links


def phs_get_link_flows(h, instance):
    n = C.c_int64()
    _chk(lib().phs_num_path_entries(h, C.c_int32(instance), C.byref(n)), "phs_num_path_entries")
    off = np.zeros(phs_num_links(h) + 1, np.int64)
    flows = np.zeros(n.value, np.int32)
    _chk(lib().phs_get_link_flows(h, C.c_int32(instance), _p(off), _p(flows), C.c_int64(n.value)), "phs_get_link_flows")
    return off, flows


def phs_get_preds(h, instance):
    n = C.c_int64()
    _chk(lib().phs_get_preds(h, C.c_int32(instance), None, None, C.c_int64(0), C.byref(n)), "phs_get_preds")
    off = np.zeros(phs_num_flows(h, instance) + 1, np.int64)
    pr = np.zeros(n.value, np.int32)
    _chk(lib().phs_get_preds(h, C.c_int32(instance), _p(off), _p(pr), C.c_int64(n.value), C.byref(n)), "phs_get_preds")
    return off, pr


def phs_get_flow_table(h, instance):
    F = phs_num_flows(h, instance)
    src, dst = np.zeros(F, np.int32), np.zeros(F, np.int32)
    b, lat = np.zeros(F, np.float64), np.zeros(F, np.float64)
    _chk(lib().phs_get_flow_table(h, C.c_int32(instance), _p(src), _p(dst), _p(b), _p(lat), C.c_int64(F)),
         "phs_get_flow_table")
    return src, dst, b, lat


def phs_get_counters(h):
    c = Counters()
    _chk(lib().phs_get_counters(h, C.byref(c)), "phs_get_counters")
    return {k: getattr(c, k) for k, _ in Counters._fields_}


def phs_instance_path(h, instance):
    return lib().phs_instance_path(h, C.c_int32(instance)).decode()


# ---------------------------------------------------------------------------------------------- convenience
class Sim:
    """Owns a phs_sim handle.  Methods forward to the C-named calls above."""

    def __init__(self, desc: dict, seed: int = 0, batch: int = 1, event_log: bool = False, path: int = 0,
                 cta_slots: int = 0, decompose: bool = True, history: int = 0, windows: bool = True):
        self.h = phs_create_topology(desc, seed, batch)
        self.batch = batch
        if event_log:
            phs_enable_event_log(self.h, True)
        if not decompose:
            phs_set_decomposition(self.h, False)
        if history:
            phs_enable_history(self.h, history)
        if not windows:
            phs_set_windows(self.h, False)
        if path or cta_slots:
            phs_set_scheduler(self.h, path, cta_slots)

    def close(self):
        if getattr(self, "h", None):
            phs_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @classmethod
    def from_workload(cls, w, event_log=False, instances=None, path=0, cta_slots=0, decompose=True, history=0,
                      windows=True):
        """Builds a batch from a workloads.Workload (optionally a subset of its instances; instance i keeps its own
        seed only if the subset is a contiguous range, so subsets are given as (first, count))."""
        first, count = (0, w.batch) if instances is None else instances
        sim = cls(w.desc, seed=w.base_seed + w.instances[first].seed, batch=count, event_log=event_log, path=path,
                  cta_slots=cta_slots, decompose=decompose, history=history, windows=windows)
        n_links = phs_num_links(sim.h)
        insts = w.instances[first:first + count]
        assert all(inst.seed == insts[0].seed + i for i, inst in enumerate(insts)), "instance seeds must be consecutive"
        from . import workloads as W
        caps = W.capacity_matrix(w.desc, insts, n_links)    # [count][n_links] if every instance overrides them
        if caps is not None and count > 1:
            phs_set_link_capacities_batch(sim.h, caps)
        else:
            for i, inst in enumerate(insts):
                cap = inst.capacities(w.desc, n_links)
                if cap is not None:
                    phs_set_link_capacities(sim.h, i, cap)
        # identical op structure across instances -> batched submission; else per instance
        same = getattr(w, "uniform_ops", False)      # the generator states it; otherwise compare
        if not same and count > 1:
            same = all(len(x.ops) == len(insts[0].ops) for x in insts) and all(
                isinstance(o, W.Coll) and o.chunks == 1 and not len(o.after_flows) for x in insts for o in x.ops)
            for k, op0 in enumerate(insts[0].ops) if same else ():
                ok = all(x.ops[k].kind == op0.kind and np.array_equal(x.ops[k].ranks, op0.ranks)
                         and tuple(x.ops[k].after) == tuple(op0.after) for x in insts)
                if not ok:
                    same = False
                    break
        if same and count > 1:
            nb, st = W.batched_sizes(w, first, count)        # host arrays [n_ops][count]
            for k, op0 in enumerate(insts[0].ops):
                phs_add_collective_batch(sim.h, op0.kind, op0.ranks, nb[k], st[k], op0.after)
        else:
            for i, inst in enumerate(insts):
                W.apply(inst,
                        lambda kind, ranks, nb, st, after, chunks=1, after_flows=(), i=i: phs_add_collective(
                            sim.h, i, kind, ranks, nb, st, after, chunks, after_flows),
                        lambda src, dst, nb, st, do, di, conn, i=i: phs_add_flows(sim.h, i, src, dst, nb, st, do, di, conn),
                        lambda gpu, dur, lane, st, do, di, i=i: phs_add_spans(sim.h, i, gpu, dur, lane, st, do, di))
        return sim

    def finalize(self, stream=None):
        phs_finalize(self.h, stream)

    def run(self, stream=None, until=None):
        if until is None:
            phs_run(self.h, stream)
        else:
            phs_run_until(self.h, until, stream)

    def run_static(self, t_done_dev=None, bneck_dev=None, stream=None):
        phs_run_static(self.h, t_done_dev, bneck_dev, self.total_flows, stream)

    def num_flows(self, i):
        return phs_num_flows(self.h, i)

    @property
    def total_flows(self):
        return phs_total_flows(self.h)

    def completion_times(self, i):
        return phs_get_completion_times(self.h, i)

    def bottlenecks(self, i):
        return phs_get_bottlenecks(self.h, i)

    def collective_times(self, i):
        return phs_get_collective_times(self.h, i)

    def event_log(self, i):
        return phs_get_event_log(self.h, i)

    def paths(self, i):
        return phs_get_paths(self.h, i)

    def link_flows(self, i):
        return phs_get_link_flows(self.h, i)

    def preds(self, i):
        return phs_get_preds(self.h, i)

    def flows(self, i):
        return phs_get_flow_table(self.h, i)

    def history(self, i):
        return phs_get_flow_history(self.h, i)

    def counters(self):
        return phs_get_counters(self.h)

    def path_of(self, i):
        return phs_instance_path(self.h, i)
