"""-m "not gpu": pins of oracle/sched_oracle.py (Algorithm 1 and the batch-metadata builder) against what the paper and
the mathematics fix: a hand-worked example in the shape of Figure 6 (tests/golden/deficit_worked_example.txt), the
amortized bound of PAPER.md:209, the idle / liveness rule, decodes never displaced,
first misfit stops the scan and arrival-time order, deficit cleared on decode-only iterations, and a
per-position brute-force check of the metadata."""
import os

import numpy as np
import pytest

import sangam_inputs as si
from oracle.sched_oracle import PAGE, SchedOracle

HERE = os.path.dirname(os.path.abspath(__file__))


def test_hand_worked_example_figure6():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "deficit_worked_example.txt")) if l.strip() and not l.startswith("#")]
    s = SchedOracle(tau=100, block=10)
    for i in range(3):                                   # three requests already decoding (never finish a block here)
        s.submit(100 + i, -1.0, 10, 10, 10)
    s.tau = 10 ** 6
    d, a = s.schedule(); s.complete([]); assert len(a) == 3
    s.tau, s.deficit = 100, 0
    for rid, tok in ((1, 40), (2, 50), (3, 120)):        # waiting prefills, arrival order p1 < p2 < p3
        s.submit(rid, float(rid), tok - 10, 10, 10)
    for t, n_dec, budget, adm, deficit in rows:
        decodes, admitted = s.schedule()
        assert len(decodes) == int(n_dec)
        assert [p.seq_len for p in admitted] == ([] if adm == "-" else [int(x) for x in adm.split(",")])
        assert s.deficit == int(deficit), (t, s.deficit)
        s.complete([0] * len(decodes))


def _drive(s, trace, iters, rng, p_done=0.3):
    """Feed a trace by iteration index (arrival = iteration), record per-iteration facts."""
    log, nxt, n = [], 0, len(trace["prompt_len"])
    for t in range(iters):
        while nxt < n and trace["arrival"][nxt] <= t:
            s.submit(nxt, float(trace["arrival"][nxt]), int(trace["prompt_len"][nxt]), int(trace["response_len"][nxt]), int(trace["output_len"][nxt]))
            nxt += 1
        waiting_before = len(s.prefills)
        deficit_before = s.deficit
        decodes, admitted = s.schedule()
        log.append(dict(t=t, D=s.block * len(decodes), A=sum(p.seq_len for p in admitted), nA=len(admitted),
                        waiting_before=waiting_before, waiting_after=len(s.prefills), S_before=deficit_before, S=s.deficit,
                        idle_admit=(len(decodes) == 0 and len(admitted) > 0 and admitted[0].seq_len > s.tau - 0 + deficit_before)))
        s.complete((rng.random(len(decodes)) < p_done).astype(int).tolist())
    return log


def _small_trace(seed, n, tau):
    g = np.random.default_rng(seed)
    return {"arrival": np.sort(g.integers(0, 3 * n, n)).astype(float), "prompt_len": g.integers(8, int(1.5 * tau), n),
            "response_len": np.full(n, 64), "output_len": g.integers(1, 64, n)}


@pytest.mark.parametrize("tau", [256, 1024])
def test_amortized_bound_over_every_busy_window(tau):
    """over a busy period of W iterations with prefills continuously waiting, admitted prefill tokens total at
    most W tau - sum D_t (the deficit is 0 when the period starts: it is cleared on decode-only iterations).  With
    D_t <= tau and no idle-rule admission the algorithm telescopes to equality minus the final carry."""
    for seed in range(6):
        s = SchedOracle(tau=tau, block=32)
        log = _drive(s, _small_trace(seed, 60, tau), 400, np.random.default_rng(seed + 100))
        w0, checked = None, 0
        for i, e in enumerate(log + [dict(waiting_before=0)]):
            busy = e["waiting_before"] > 0
            if busy and w0 is None:
                w0 = i
            if not busy and w0 is not None:
                win = log[w0:i]
                if all(x["D"] <= tau for x in win) and not any(x["idle_admit"] for x in win) and win[0]["S_before"] == 0:
                    W, sumD, sumA = len(win), sum(x["D"] for x in win), sum(x["A"] for x in win)
                    assert sumA <= W * tau - sumD
                    assert sumA == W * tau - sumD - win[-1]["S"]          # exact: nothing is lost but the final carry
                    for k in range(1, W + 1):                             # and every prefix of the busy period
                        assert sum(x["A"] for x in win[:k]) <= k * tau - sum(x["D"] for x in win[:k])
                    checked += 1
                w0 = None
        assert checked > 0


def test_idle_rule_gives_liveness_and_only_when_idle():
    s = SchedOracle(tau=100, block=10)
    s.submit(1, 0.0, 990, 10, 10)                      # 1000 tokens >> tau
    d, a = s.schedule()
    assert [p.rid for p in a] == [1] and s.deficit == 0   # admitted into the idle system; budget went negative -> 0
    s.complete([])
    s.submit(2, 1.0, 240, 10, 10)                      # 250 tokens: with one decode in flight it must wait for carry
    waits = 0
    while True:
        d, a = s.schedule()
        assert [r.rid for r in d] == [1]
        s.complete([0])
        if a:
            break
        waits += 1
    assert waits == 2                                   # budgets 90, 180, 270 >= 250 on the third iteration


def test_decodes_are_never_displaced_even_above_the_budget():
    s = SchedOracle(tau=64, block=32)
    for i in range(5):
        s.submit(i, 0.0, 8, 32, 32)
    s.tau = 10 ** 6
    s.schedule(); s.complete([])
    s.tau, s.deficit = 64, 0                            # 5 decodes = 160 tokens > tau
    s.submit(9, 1.0, 8, 32, 32)
    d, a = s.schedule()
    assert len(d) == 5 and a == [] and s.deficit == 0   # all decodes seated, no prefill, nothing carried


def test_first_misfit_stops_the_scan_and_arrival_order():
    s = SchedOracle(tau=100, block=10)
    s.submit(1, 0.0, 10, 20, 20)                        # 30 tokens, will decode two blocks
    s.schedule(); s.complete([])
    s.submit(2, 5.0, 490, 10, 10)                       # 500 tokens: does not fit
    s.submit(3, 6.0, 10, 10, 10)                        # 20 tokens: would fit, but comes later
    d, a = s.schedule()
    assert a == [] and [e[2].rid for e in s.prefills] == [2, 3]
    s.complete([1])                                     # request 1 resolves block 0 -> its re-prefill (arrival 0.0) queues
    assert [e[2].rid for e in s.prefills] == [1, 2, 3]  # older request's re-prefill ahead of newer fresh prefills
    d, a = s.schedule()
    assert [p.rid for p in a] == [1]                    # 30 tokens fit; request 2 (500 > 230 left) still blocks request 3


def test_deficit_cleared_on_decode_only_iteration():
    s = SchedOracle(tau=100, block=10)
    s.submit(1, 0.0, 10, 10, 10)
    s.schedule()
    assert s.deficit == 80
    s.complete([])
    s.schedule()                                        # nothing waiting
    assert s.deficit == 0


def test_memory_blocked_head_stops_the_scan_and_pages_are_conserved():
    s = SchedOracle(tau=10 ** 6, block=32, num_pages=10)
    s.submit(1, 0.0, 64, 32, 32)                        # 6 pages
    s.submit(2, 1.0, 64, 32, 32)                        # 6 pages: does not fit next to request 1
    s.submit(3, 2.0, 16, 16, 16)                        # 2 pages: would fit, but the head blocks it
    d, a = s.schedule()
    assert [p.rid for p in a] == [1] and len(s.free_pages) == 4
    s.complete([])
    d, a = s.schedule(); assert a == []
    s.complete([1])                                     # request 1 retires
    assert len(s.free_pages) == 10
    d, a = s.schedule()
    assert [p.rid for p in a] == [2, 3] and len(s.free_pages) == 2


def test_metadata_against_a_per_position_construction():
    tr = si.sched_trace(3, 12, qps=50.0, kind="sharegpt_like")
    s = SchedOracle(tau=4096, block=32, num_pages=4096)
    for i in range(12):
        s.submit(i, float(tr["arrival"][i]), int(tr["prompt_len"][i]), int(tr["response_len"][i]), int(tr["output_len"][i]))
    rng = np.random.default_rng(0)
    seen_mixed = False
    for it in range(30):
        decodes, admitted = s.schedule()
        W = 4096 // PAGE
        cu, ctx, bt, sm, rid, nd = s.metadata(W)
        assert nd == len(decodes) and len(rid) == len(decodes) + len(admitted)
        seen_mixed |= bool(decodes) and bool(admitted)
        k = 0
        for i, r in enumerate(decodes + admitted):
            assert ctx[i] == r.prompt_len + r.response_len
            rows = range(r.prompt_len + r.cur_block * 32, r.prompt_len + r.cur_block * 32 + 32) if i < nd else range(r.seq_len)
            assert cu[i + 1] - cu[i] == len(rows)
            for pos in rows:                               # brute force, one position at a time
                assert sm[k] == r.pages[pos // PAGE] * PAGE + pos % PAGE
                k += 1
            assert list(bt[i, :len(r.pages)]) == r.pages and np.all(bt[i, len(r.pages):] == -1)
        assert k == len(sm) and len(set(sm.tolist())) == len(sm)         # slots unique within one iteration (reading S11)
        owned = [pg for r in s.reqs.values() if r.pages for pg in r.pages]
        assert len(set(owned)) == len(owned) and len(owned) + len(s.free_pages) == 4096
        s.complete((rng.random(len(decodes)) < 0.4).astype(int).tolist())
    assert seen_mixed


def test_trace_generator_matches_table1_statistics():
    for kind, (pm, p99, om, o99, resp) in si.TRACE_STATS.items():
        tr = si.sched_trace(0, 20000, 5.0, kind)
        assert abs(np.median(tr["prompt_len"]) / pm - 1) < 0.05 and abs(np.median(tr["output_len"]) / om - 1) < 0.06
        assert abs(np.percentile(tr["output_len"], 99) / o99 - 1) < 0.12
        assert np.all(tr["prompt_len"] + tr["output_len"] <= 4096) and np.all(tr["response_len"] == resp)
