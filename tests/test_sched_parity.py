"""-m "not gpu": the product's scheduler (sangam_sched_*, C++ behind the C ABI) against oracle/sched_oracle.py on seeded
arrival traces with Table-1-like length statistics: every integer it produces -- who is in the
microbatch, the deficit, cu_q_lens, ctx_lens, block_table, slot_mapping -- must be identical, iteration by iteration."""
import numpy as np
import pytest

import paper_2607_04206_b200 as sg
import sangam_inputs as si
from oracle.sched_oracle import SchedOracle


def _run(tau, kind, qps, n, iters, num_pages, max_batch, max_total_q, seed, iter_time=0.05):
    tr = si.sched_trace(seed, n, qps, kind)
    W = 4096 // 16 + 64 + 8
    prod = sg.Scheduler(tau=tau, num_pages=num_pages, max_batch=max_batch, max_total_q=max_total_q, max_pages_per_req=W)
    orc = SchedOracle(tau=tau, block=32, num_pages=num_pages, max_batch=max_batch, max_total_q=max_total_q)
    steps_left = {}
    nxt, mixed, busy_windows = 0, 0, 0
    for it in range(iters):
        now = it * iter_time
        while nxt < n and tr["arrival"][nxt] <= now:
            a = (nxt, float(tr["arrival"][nxt]), int(tr["prompt_len"][nxt]), int(tr["response_len"][nxt]), int(tr["output_len"][nxt]))
            assert prod.submit(*a) == 0
            orc.submit(*a)
            nxt += 1
        b = prod.next()
        decodes, admitted = orc.schedule()
        cu, ctx, bt, sm, rid, nd = orc.metadata(W)
        R = len(rid)
        assert (b.batch, b.num_decodes, b.total_q, b.deficit) == (R, nd, int(cu[-1]), orc.deficit), f"iteration {it}"
        assert np.array_equal(prod.arrays["req_ids"][:R], rid)
        assert np.array_equal(prod.arrays["cu_q_lens"][:R + 1], cu)
        assert np.array_equal(prod.arrays["ctx_lens"][:R], ctx)
        assert np.array_equal(prod.arrays["block_table"][:R], bt)
        assert np.array_equal(prod.arrays["slot_mapping"][:b.num_new_tokens], sm)
        assert prod.query(1) == len(orc.prefills) and prod.query(2) == len(orc.decodes) and prod.query(3) == len(orc.free_pages)
        mixed += int(nd > 0 and R > nd)
        # denoising steps per block come from the trace (stand-in for confidence-threshold unmasking)
        done = []
        for r in decodes:
            key = (r.rid, r.cur_block)
            steps_left.setdefault(key, int(tr["steps"][r.rid, r.cur_block]))
            steps_left[key] -= 1
            done.append(1 if steps_left[key] <= 0 else 0)
        prod.complete(done)
        orc.complete(done)
    assert nxt > n // 2
    return mixed


@pytest.mark.parametrize("tau", [512, 1024, 2048, 16384])          # the budgets of PAPER.md:327
@pytest.mark.parametrize("kind", ["sharegpt_like", "arxiv_like"])
def test_product_equals_oracle_on_seeded_traces(tau, kind):
    mixed = _run(tau, kind, qps=6.0, n=160, iters=900, num_pages=6000, max_batch=64, max_total_q=20000, seed=tau + len(kind))
    assert mixed > 0, "the trace never produced a hybrid (decodes + prefills) microbatch"


def test_product_equals_oracle_under_memory_and_capacity_pressure():
    # a pool that holds only a handful of requests and a batch cap that binds: the memory / capacity readings (S21, S22)
    _run(1024, "sharegpt_like", qps=20.0, n=120, iters=1500, num_pages=700, max_batch=6, max_total_q=6000, seed=9)


def test_submit_rejects_what_can_never_run():
    s = sg.Scheduler(tau=1024, num_pages=100, max_batch=4, max_total_q=1000, max_pages_per_req=32)
    assert s.submit(1, 0.0, 2000, 64, 64) == -3          # more tokens than max_total_q / pages than the block table
    assert s.submit(2, 0.0, 100, 64, 64) == 0
    assert s.submit(2, 1.0, 100, 64, 64) == -1           # duplicate id
    assert s.submit(3, 0.0, 100, 0, 1) == -1
    b = s.next()
    assert b.batch == 1 and b.num_decodes == 0
    with pytest.raises(sg.SangamError):
        s.next() if False else s.complete([1])           # n != number of decodes of the last batch
