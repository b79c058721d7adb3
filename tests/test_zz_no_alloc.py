"""-m gpu: sangam_confidence_sample_static, the sampler entry point that allocates nothing (its scratch is a static device
array inside libsangam.so), against the existing sangam_confidence_sample on the same inputs, two calls in a row -- the
second with a different batch, so that it finds the first call's partials in the shared array.  Collected last on purpose
(the file name sorts after every other test file): the suite runs with pytest -x."""
import numpy as np
import pytest

import sangam_inputs as si
from gpu_harness import t_bf16, t_i32

pytestmark = pytest.mark.gpu


def _inputs(seed, vocab, rows_per_req):
    g = np.random.default_rng(seed)
    rows = int(sum(rows_per_req))
    x = 2.0 * g.standard_normal((rows, vocab), dtype=np.float32)
    x[np.arange(rows), g.integers(0, vocab, rows)] += g.choice([0.0, 6.0, 12.0, 20.0], rows)      # flat to very confident rows
    masked = (g.random(rows) < 0.7).astype(np.int32)
    cu = np.concatenate([[0], np.cumsum(rows_per_req)]).astype(np.int32)
    return si.f32_to_bf16_bits(x), masked, cu


def _outputs(rows):
    import torch
    return (torch.full((rows,), -1, dtype=torch.int32, device="cuda"), torch.full((rows,), -1.0, dtype=torch.float32, device="cuda"),
            torch.full((rows,), -1, dtype=torch.int32, device="cuda"))


def test_static_sampler_matches_the_allocating_one_on_two_calls_in_a_row():
    import torch
    import paper_2607_04206_b200 as sg
    thr = 0.9
    # call 1: 3 x 32 rows at LLaDA's vocabulary (many slices per row); call 2: 40 ragged rows at a small vocabulary
    # (other slicing, fewer partials: stale entries of call 1 stay in the array and must not be read)
    for seed, vocab, rows_per_req in ((5, 126464, [32, 32, 32]), (6, 1000, [7, 1, 32])):
        logits, masked, cu = _inputs(seed, vocab, rows_per_req)
        rows = logits.shape[0]
        d_logits, d_masked, d_cu = t_bf16(logits), t_i32(masked), t_i32(cu)
        eng = sg.Sangam(num_q_heads=4, num_kv_heads=4, head_dim=64, num_pages=8, max_batch=len(rows_per_req), max_total_q=rows,
                        max_pages_per_req=4)
        tok_a, conf_a, un_a = _outputs(rows)
        eng.confidence_sample(d_logits, d_masked, d_cu, thr, tok_a, conf_a, un_a)
        tok_s, conf_s, un_s = _outputs(rows)
        sg.confidence_sample_static(d_logits, d_masked, d_cu, thr, tok_s, conf_s, un_s)
        torch.cuda.synchronize()
        assert torch.equal(tok_s, tok_a), "argmax differs"
        ca, cs = conf_a.cpu().numpy().astype(np.float64), conf_s.cpu().numpy().astype(np.float64)
        assert np.all(cs > 0)
        assert np.allclose(cs, ca, rtol=2e-5, atol=1e-9)          # the tolerance of tests/test_gpu_neighbours.py
        # unmask decisions: equal wherever the confidence is not within rounding of the threshold (same rule as the oracle test)
        un_a_h, un_s_h = un_a.cpu().numpy(), un_s.cpu().numpy()
        clear = np.abs(ca - thr) > 1e-4
        for r in range(len(rows_per_req)):
            lo, hi = cu[r], cu[r + 1]
            if np.all(clear[lo:hi]):
                assert np.array_equal(un_s_h[lo:hi], un_a_h[lo:hi]), f"request {r}"
        assert np.all(un_s_h[masked == 0] == 0)
        print(f"static sampler V={vocab}: {rows} rows, conf max rel diff {np.max(np.abs(cs - ca) / ca):.2e}, {int(un_s_h.sum())} unmasked")


def test_static_sampler_rejects_sizes_beyond_its_scratch_and_launches_nothing():
    import torch
    import paper_2607_04206_b200 as sg
    rows = sg.STATIC_SAMPLER_MAX_ROWS + 1
    logits = torch.zeros((rows, 8), dtype=torch.bfloat16, device="cuda")
    masked = torch.ones(rows, dtype=torch.int32, device="cuda")
    cu = torch.tensor([0, rows], dtype=torch.int32, device="cuda")
    tok, conf, un = _outputs(rows)
    with pytest.raises(sg.SangamError, match="SANGAM_STATIC_SAMPLER_MAX_ROWS"):
        sg.confidence_sample_static(logits, masked, cu, 0.9, tok, conf, un)
    torch.cuda.synchronize()
    assert int(tok.max()) == -1 and int(un.max()) == -1          # outputs untouched
    # the maximum itself is accepted
    rows = sg.STATIC_SAMPLER_MAX_ROWS
    x = torch.zeros((rows, 16), dtype=torch.bfloat16, device="cuda")
    x[:, 3] = 8.0
    tok, conf, un = _outputs(rows)
    sg.confidence_sample_static(x, masked[:rows].contiguous(), torch.tensor([0, rows], dtype=torch.int32, device="cuda"), 0.9, tok, conf, un)
    torch.cuda.synchronize()
    assert int(tok.min()) == 3 and int(tok.max()) == 3 and int(un.min()) == 1
