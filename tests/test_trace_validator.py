"""NEXT-1: trace validator.  CPU part pins oracle.validator.validate_index and the trace generator;
GPU part compares rc_validate_trace with the oracle on valid streams and on every control class
(P:L463)."""
import numpy as np
import pytest

from oracle import validator as V
import trace_inputs as T


def test_validate_index_is_the_first_position_whose_prefix_is_rejected():
    ev = T.make_trace(60, 4)
    assert V.validate_index(ev) == (True, -1) and V.validate(ev)[0]
    for kind in T.TRACE_MUTATIONS:
        m = T.mutate_trace(ev, kind, 1)
        ok, i = V.validate_index(m)
        assert not ok and not V.validate(m)[0], kind
        assert V.validate(m[:i])[0] and not V.validate(m[: i + 1])[0], kind     # brute-force prefix property


def test_generated_traces_keep_per_claim_order_and_carry_both_paths():
    ev = T.make_trace(500, 9)
    cids = np.unique(ev["claim_id"])
    fails = sum(V.failure_outcome_gate(ev, int(c)) for c in cids[:40])
    obs = sum(V.observation_gate(ev, int(c)) for c in cids[:40])
    assert fails > 0 and obs > 0 and fails + obs <= 40


@pytest.mark.gpu
@pytest.mark.parametrize("seed", [0, 1])
def test_gpu_validator_matches_oracle_on_valid_and_mutated_streams(seed):
    from paper_2606_01387_b200 import rc
    ev = T.make_trace(3000, seed)
    rep, claims = rc.validate_trace(ev)
    assert rep["ok"] == 1 and rep["first_bad_index"] == rc.NO_BAD and rep["n_events"] == ev.size
    assert rep["n_claims"] == np.unique(ev["claim_id"]).size == claims.size
    assert sorted(claims["claim_id"]) == sorted(np.unique(ev["claim_id"]))
    assert int(claims["n_events"].sum()) == ev.size
    for kind in T.TRACE_MUTATIONS:
        for ms in range(3):
            m = T.mutate_trace(ev, kind, 10 * seed + ms)
            ok, i = V.validate_index(m)
            rep, claims = rc.validate_trace(m)
            assert (rep["ok"] == 1) == ok and not ok, kind
            assert rep["first_bad_index"] == i, (kind, rep["first_bad_index"], i)
            assert rep["n_failure_gate"] == 0 and rep["n_observation_gate"] == 0     # gates presuppose a valid stream


@pytest.mark.gpu
def test_gpu_validator_gates_per_claim_match_oracle():
    from paper_2606_01387_b200 import rc
    ev = T.make_trace(250, 7)
    rep, claims = rc.validate_trace(ev)
    nf = no = 0
    for c in claims:
        cid = int(c["claim_id"])
        f, o = V.failure_outcome_gate(ev, cid), V.observation_gate(ev, cid)
        assert bool(c["gates"] & rc.GATE_FAILURE) == f and bool(c["gates"] & rc.GATE_OBSERVATION) == o, hex(cid)
        nf += f
        no += o
    assert rep["n_failure_gate"] == nf and rep["n_observation_gate"] == no and nf > 0 and no > 0


@pytest.mark.gpu
def test_gpu_validator_edge_cases_and_scale():
    from paper_2606_01387_b200 import rc
    rep, claims = rc.validate_trace(np.zeros(0, rc.EVENT_DTYPE))
    assert rep["ok"] == 1 and rep["n_claims"] == 0
    one = np.zeros(1, rc.EVENT_DTYPE)
    one["claim_id"], one["code"] = 5, 2                   # MATERIALIZED before ACCEPTED: post-hoc naming
    rep, _ = rc.validate_trace(one)
    assert rep["ok"] == 0 and rep["first_bad_index"] == 0 and V.validate_index(one) == (False, 0)
    big = T.make_trace(100000, 3)                         # ~0.9 M events: properties that hold at any size
    rep, claims = rc.validate_trace(big)
    assert rep["ok"] == 1 and rep["n_claims"] == np.unique(big["claim_id"]).size
    n_ref = int((big["code"] == 8).sum())
    assert rep["n_failure_gate"] == n_ref                 # every refused claim of a valid generated stream took path B
    m = T.mutate_trace(big, "wrong_claim", 2)
    rep, _ = rc.validate_trace(m, want_claims=False)
    assert rep["ok"] == 0 and (False, rep["first_bad_index"]) == V.validate_index(m)


def test_real_stream_from_the_oracle_run_validates_both_ways():
    from conftest import build_tiny_oracle
    o, wl, wave, pool, fill = build_tiny_oracle()
    ids = [c.claim_id for c in wl.claims]
    o.accept(ids, [c.P for c in wl.claims], [c.N for c in wl.claims], wave.bt_off, wave.bt_ids)
    o.materialize(ids); o.offload(ids); o.set_faults(wave.faults); o.restore(ids)
    ev = o.outcomes()
    assert V.validate_index(ev) == (True, -1)


def test_request_traces_validate_and_every_request_mutation_is_rejected():
    ev, runs = T.make_request_trace(120, 2)
    assert V.validate_index(ev) == (True, -1) and len(runs) > 20
    assert {9, 10} <= set(int(c) for c in ev["code"])
    for kind in T.REQUEST_MUTATIONS:
        m = T.mutate_request_trace(ev, runs, kind, 1)
        ok, i = V.validate_index(m)
        assert not ok and V.validate(m[:i])[0], kind


@pytest.mark.gpu
@pytest.mark.parametrize("seed", [0, 3])
def test_gpu_validator_request_runs_and_policies_match_oracle(seed):
    """NEXT-3 on the validator: demotion / expiry transitions and the cross-claim rule for request-level
    refusal runs (exact failed subset, contiguous, one request id) -- P:L87."""
    from paper_2606_01387_b200 import rc
    ev, runs = T.make_request_trace(1500, seed)
    rep, claims = rc.validate_trace(ev)
    assert rep["ok"] == 1 and rep["first_bad_index"] == rc.NO_BAD
    n_ref = len({int(e["claim_id"]) for e in ev if int(e["code"]) == 8})
    assert rep["n_failure_gate"] == n_ref and rep["n_observation_gate"] == int((ev["code"] == 6).sum())
    for kind in T.REQUEST_MUTATIONS:
        for ms in range(4):
            m = T.mutate_request_trace(ev, runs, kind, 10 * seed + ms)
            ok, i = V.validate_index(m)
            rep, _ = rc.validate_trace(m, want_claims=False)
            assert not ok and rep["ok"] == 0 and rep["first_bad_index"] == i, (kind, ms, rep["first_bad_index"], i)
    both = np.concatenate([T.make_trace(800, seed), ev])          # per-claim refusals and request runs in one stream
    both["seq"] = np.arange(both.size)
    rep, _ = rc.validate_trace(both, want_claims=False)
    assert rep["ok"] == 1 and V.validate_index(both) == (True, -1)


def test_pressure_traces_validate_and_every_pressure_mutation_is_rejected():
    """NEXT-3 allocator side: victim demotions and protected-conflict refusal runs."""
    ev, runs = T.make_pressure_trace(150, 1)
    assert V.validate_index(ev) == (True, -1) and len(runs) > 20
    assert int(((ev["code"] == 9) & (ev["arg"] != 0)).sum()) > 50 and int(((ev["code"] == 9) & (ev["arg"] == 0)).sum()) > 5
    for kind in T.PRESSURE_MUTATIONS:
        for ms in range(3):
            m = T.mutate_pressure_trace(ev, runs, kind, ms)
            ok, i = V.validate_index(m)
            assert not ok and V.validate(m[:i])[0], (kind, ms)


@pytest.mark.gpu
@pytest.mark.parametrize("seed", [0, 5])
def test_gpu_validator_pressure_traces_match_oracle(seed):
    from paper_2606_01387_b200 import rc
    ev, runs = T.make_pressure_trace(1200, seed)
    rep, claims = rc.validate_trace(ev)
    assert rep["ok"] == 1 and rep["first_bad_index"] == rc.NO_BAD and V.validate_index(ev) == (True, -1)
    for kind in T.PRESSURE_MUTATIONS:
        for ms in range(4):
            m = T.mutate_pressure_trace(ev, runs, kind, 10 * seed + ms)
            ok, i = V.validate_index(m)
            rep, _ = rc.validate_trace(m, want_claims=False)
            assert not ok and rep["ok"] == 0 and rep["first_bad_index"] == i, (kind, ms, rep["first_bad_index"], i)


@pytest.mark.gpu
def test_gpu_validator_orders_a_claim_with_many_events():
    """one claim with a very long event run (tv_walk sorts its bucket with a heap sort, not O(c^2))."""
    from paper_2606_01387_b200 import rc
    n = 300000
    ev = np.zeros(n + 2, rc.EVENT_DTYPE)
    ev["claim_id"] = 77
    ev["code"] = 100                                       # USE, USE, ... after ACCEPTED, MATERIALIZED
    ev["code"][0], ev["code"][1] = 1, 2
    ev["seq"] = np.arange(n + 2)
    rep, claims = rc.validate_trace(ev)
    assert rep["ok"] == 1 and rep["n_claims"] == 1 and int(claims[0]["n_events"]) == n + 2
    ev["code"][n // 2] = 3                                 # OFFLOADED in the middle: the next USE is restore-after-use
    rep, _ = rc.validate_trace(ev, want_claims=False)
    assert rep["ok"] == 0 and rep["first_bad_index"] == n // 2 + 1 == V.validate_index(ev[: n // 2 + 2])[1]
