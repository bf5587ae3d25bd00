"""phs_run_static (include/phs.h): the run that allocates nothing -- the grid kernel with its scratch in the library's
fixed __device__ array -- against the existing path (phs_run) on the same handle-building inputs.  The file is named
so that pytest collects it last.  Bar: the one of tests/test_gpu_parity.py (completion times within 1e-9 relative, and
in fact bit-equal; bottleneck ids exact).  Two calls in a row share the array; both must be right."""
import numpy as np
import pytest

from paper_2505_01616_b200 import binding as B
from paper_2505_01616_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _existing_path(w, **kw):
    sim = B.Sim.from_workload(w, **kw)
    sim.run()
    t = np.concatenate([sim.completion_times(i) for i in range(w.batch)])
    b = np.concatenate([sim.bottlenecks(i) for i in range(w.batch)])
    ct = [sim.collective_times(i) for i in range(w.batch)]
    sim.close()
    return t, b, ct


def _static_run(sim):
    import torch
    n = sim.total_flows
    t = torch.full((n,), -1.0, dtype=torch.float64, device="cuda")
    b = torch.full((n,), -7, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    sim.run_static(t.data_ptr(), b.data_ptr())
    return t.cpu().numpy(), b.cpu().numpy()


def _assert_same(t, b, t_ref, b_ref):
    assert not np.isnan(t).any()
    np.testing.assert_allclose(t, t_ref, rtol=1e-9, atol=0)        # the stated bar
    assert np.array_equal(t, t_ref), "completion times are expected to be bit-equal"
    assert np.array_equal(b, b_ref)


def test_static_run_equals_the_existing_path_on_two_calls_in_a_row():
    # call 1: several decomposed units of ring traffic, one after the other through the array
    w1 = W.cfg1(batch=3, n_hosts=8, gph=4, n_leaves=4, n_spines=2)
    # call 2: one unit with many concurrent flows and many filling rounds per event -- a different layout of the array,
    # larger than call 1's, so whatever call 1 left behind lies inside it
    w2 = W.cfg4(batch=2, n_hosts=8, gph=8, n_leaves=4, n_spines=2)
    ref1, ref2 = _existing_path(w1), _existing_path(w2)
    s1, s2 = B.Sim.from_workload(w1), B.Sim.from_workload(w2)
    s1.finalize()
    s2.finalize()
    t, b = _static_run(s1)
    _assert_same(t, b, ref1[0], ref1[1])
    assert s1.path_of(0) == "grid" and s1.counters()["grid_ctas"] >= 1
    for i in range(w1.batch):                                      # the handle holds the same results
        assert np.array_equal(s1.collective_times(i), ref1[2][i])
    t, b = _static_run(s2)
    _assert_same(t, b, ref2[0], ref2[1])
    # and back: the smaller layout again, now over call 2's leftovers; then the handle's ordinary run still works
    t, b = _static_run(s1)
    _assert_same(t, b, ref1[0], ref1[1])
    s1.run()
    assert np.array_equal(np.concatenate([s1.completion_times(i) for i in range(w1.batch)]), ref1[0])
    s1.close()
    s2.close()


def test_static_run_limits_and_states():
    # larger than the static array: refused with a clear error, nothing ran
    d = W.topo_desc(W.TOPO_SINGLE, 60, 8)                          # 480 GPUs: 229,920 concurrent flows, 9.2 MB of state
    sim = B.Sim(d, batch=1)
    B.phs_add_collective(sim.h, 0, B.ALLTOALL, np.arange(480, dtype=np.int32), 480e6)
    sim.finalize()
    with pytest.raises(B.PhsError) as e:
        sim.run_static()
    assert e.value.code == B.PHS_ERANGE and "static scratch holds" in str(e.value)
    sim.close()
    # more units than the static list holds
    w = W.cfg3(batch=600)                                          # 9 units per instance
    sim = B.Sim.from_workload(w)
    sim.finalize()
    with pytest.raises(B.PhsError) as e:
        sim.run_static()
    assert e.value.code == B.PHS_ERANGE and "unit list" in str(e.value)
    sim.close()
    # not finalized / event log on: wrong state
    w = W.cfg0()
    sim = B.Sim.from_workload(w)
    with pytest.raises(B.PhsError) as e:
        sim.run_static()
    assert e.value.code == B.PHS_ESTATE
    sim.close()
    sim = B.Sim.from_workload(w, event_log=True)
    sim.finalize()
    with pytest.raises(B.PhsError) as e:
        sim.run_static()
    assert e.value.code == B.PHS_ESTATE
    sim.close()
    # outputs are optional; an empty batch member is fine
    sim = B.Sim.from_workload(w)
    sim.finalize()
    sim.run_static()
    ref = _existing_path(w)
    assert np.array_equal(sim.completion_times(0), ref[0]) and np.array_equal(sim.bottlenecks(0), ref[1])
    sim.close()
