"""Mutation check of the oracle's pins: every mutant below is a plausible mistake in oracle/orc_netsim.c (a dropped
term, a wrong index, a wrong sign); each is applied to a scratch copy, built, and tests/test_oracle_pins.py is run
against it through ORC_LIB_PATH.  The pins must FAIL for every mutant (VERDICT r1 "What's weak" #1 lists the three
that used to survive: M1, M2, M3, plus the hash-lane mutant M4)."""
import os
import subprocess
import sys
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "orc_netsim.c")

# (name, text in orc_netsim.c, replacement, -k expression selecting pins that should catch it (speed only))
MUTANTS = [
    ("M1_release_ignores_start", "double st = s->start[g] > now ? s->start[g] : now;", "double st = now;",
     "dependent_flow"),
    ("M2_no_clamp", "return r > 0.0 ? r : 0.0;", "return r;", "q11"),
    ("M3_sum_lam_doubled", "s->work[4] += lam;", "s->work[4] += 2 * lam;", "work_counters"),
    ("M4_down_lane_low_bits", "pd = (int32_t)((H >> 32) % (uint64_t)P);", "pd = (int32_t)(H % (uint64_t)P);",
     "down_lane"),
    ("M5_no_fifo_pred", "if (push_pred(s, first + (st - 1) * N + i)) return ORC_ENOMEM;               /* sender FIFO */",
     "", "ring_dag"),
    ("M6_no_received_edge", "if (push_pred(s, last + (ia + A->n - 1) % A->n)) return -1; /* received by rho */", "",
     "after_chains or mixed_kind"),
    ("M7_tie_to_highest_id", "int64_t sh = w->cap_rem[l] / w->n[l];\n        if (b < 0 || sh < s) { b = l; s = sh; }",
     "int64_t sh = w->cap_rem[l] / w->n[l];\n        if (b < 0 || sh <= s) { b = l; s = sh; }", "p1_lone or p3_cfg0"),
    ("M8_no_latency_on_release", "t_act[g] = st + s->Lat[g];", "t_act[g] = st;", "p2_uniform or input_validation"),
    ("M9_a2a_after_edges_to_rho_dropped",
     "if (push_pred(s, A->first_flow + x * (A->n - 1) + (ia < x ? ia : ia - 1))) return -1;", "",
     "mixed_kind or alltoall_after"),
    ("M10_sum_R_counts_events", "s->work[2] += R;", "s->work[2] += 1;", "work_counters"),
    ("M11_settle_sign", "double r = rem - m;", "double r = rem + m;", "p6 or q11"),
    ("M12_chunk_not_divided", "} else if (kind <= ORC_REDUCESCATTER_RING) {\n    double chunk = bytes / (double)N;",
     "} else if (kind <= ORC_REDUCESCATTER_RING) {\n    double chunk = bytes;", "p2_uniform"),
    ("M13_chain_no_fifo", "if (ch > 0 && push_pred(s, first + (ch - 1) * (N - 1) + i)) return ORC_ENOMEM; /* sender FIFO */",
     "", "next3_pipelined"),
    ("M14_tree_root_waits_for_one_child", "if (N > 2 && push_pred(s, first + ch * per + 1)) return ORC_ENOMEM;", "",
     "next3_tree"),
    ("M16_rollback_completion_time_from_now", "tc[f] = t_last[f] + q;", "tc[f] = now + q;", "next1"),
    ("M17_rollback_ignores_latest_predecessor", "if (s->done_ev[p] >= 0) { if (s->t_done[p] > latest) latest = s->t_done[p]; }",
     "if (s->done_ev[p] >= 0) { }", "next1"),
    ("M18_rollback_keeps_the_event_at_T", "while (k < s->n_ev && s->ev[k].t < T) k++;",
     "while (k < s->n_ev && s->ev[k].t <= T) k++;", "next1"),
    ("M15_chain_after_ignores_last_chunk", "for (int32_t f = A->first_flow + (A->chunks - 1) * per_chunk;",
     "for (int32_t f = A->first_flow;", "next3_after"),
]


@pytest.mark.parametrize("name,old,new,select", MUTANTS, ids=[m[0] for m in MUTANTS])
def test_pins_kill_mutant(name, old, new, select):
    src = open(SRC).read()
    assert src.count(old) == 1, f"mutant {name} no longer applies (text not found exactly once)"
    with tempfile.TemporaryDirectory() as tmp:
        c = os.path.join(tmp, "orc_mut.c")
        so = os.path.join(tmp, "liborc_mut.so")
        with open(c, "w") as f:
            f.write(src.replace(old, new))
        subprocess.check_call(["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fno-fast-math", "-w", "-fPIC", "-shared",
                               "-I", os.path.join(ROOT, "oracle"), c, "-o", so, "-lm"])
        env = dict(os.environ, ORC_LIB_PATH=so)
        r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_oracle_pins.py"), "-x", "-q",
                            "-k", select, "-p", "no:cacheprovider"], env=env, cwd=ROOT, capture_output=True, text=True)
        assert r.returncode == 1, f"mutant {name} survived the pins:\n{r.stdout[-2000:]}"
