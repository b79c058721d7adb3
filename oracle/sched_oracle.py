"""Plain Python restatement of the paper's worker-level scheduler and of the batch metadata it hands to the kernels.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py): imported by tests/ and by bench.py's CPU legs; it shares no code with
the product's scheduler (paper_2607_04206_b200/csrc/sched.cu) and neither imports the other.

What it follows, step by step and in the paper's notation:
  * Algorithm 1 "Deficit token-budget scheduling" (the listing lost its line numbers 3 and 5-8 and
    split its arrows -- reading S19 of DESIGN.md -- the prose of PAPER.md:166 and PAPER.md:205-207 fills them in):
        if prefills is empty:  deficit <- 0;  return decodes                      (decode-only iteration)
        budget <- tau - Tokens(decodes) + deficit
        microbatch <- decodes                                                     (decodes are never displaced)
        while prefills is not empty:
            p <- first request in prefills                                        (arrival-time order)
            idle <- (microbatch is empty)
            if Tokens(p) <= budget or idle:  move p into microbatch;  budget <- budget - Tokens(p)
            else: break                                                           (p waits; prefills cannot be split)
        deficit <- max(budget, 0)
        return microbatch
  * queue order: "arrival-time order, not strict FIFO, so a re-prefill from an older request is ordered ahead of a fresh
    prefill from a newer one"; ties are broken by submission order (reading S20).
  * Tokens(decode) = one response block (32; "a decode contributes an entire response block");
    Tokens(prefill) = prompt + response region, the whole sequence.
  * request life cycle (Fast-dLLM style caching): prefill -> decode block 0 for some
    denoising steps -> at the block boundary the cache is recomputed: a re-prefill of the whole sequence, queued with
    the request's ORIGINAL arrival time -> decode block 1 -> ... for ceil(output_len / block) blocks.
  * capacities (reading S22): a head prefill that would exceed the batch arrays (max_batch requests, max_total_q rows)
    does not fit either.
  * memory (reading S21; the paper only says "when memory capacity is also available"): a request's pages
    are taken at its first admission; if the pool cannot hold it, the head prefill "does not fit" and stops the scan
    like any other misfit -- except under the idle rule, where nothing can be done and the scan also stops.
  * batch metadata: requests in microbatch order (decodes first, then prefills);
    a decode's q rows are its current block, a prefill's its whole sequence; ctx = prompt + response for both;
    slot = page * 16 + offset of every K/V row the iteration produces (the decode's block, the prefill's sequence).
"""
from __future__ import annotations

import numpy as np

PAGE = 16


class Request:
    def __init__(self, rid, arrival, prompt_len, response_len, output_len, block):
        self.rid, self.arrival = rid, arrival
        self.prompt_len, self.response_len, self.block = prompt_len, response_len, block
        self.nblocks = max(1, -(-min(output_len, response_len) // block))   # blocks past the committed EOS are never denoised
        self.cur_block = 0
        self.pages = None            # page ids once admitted

    @property
    def seq_len(self):
        return self.prompt_len + self.response_len


class SchedOracle:
    def __init__(self, tau, block=32, num_pages=1 << 20, max_batch=None, max_total_q=None):
        self.tau, self.block = int(tau), int(block)
        self.max_batch, self.max_total_q = max_batch, max_total_q       # capacities of the batch arrays (reading S22)
        self.deficit = 0
        self.decodes = []            # in-flight decodes, in the order they became decodes
        self.prefills = []           # waiting prefills: (arrival, seq_no, request)
        self.free_pages = list(range(num_pages - 1, -1, -1))     # stack: pop() yields 0, 1, 2, ...
        self.seq = 0
        self.reqs = {}
        self.last = ([], [])

    # ---- queue maintenance -----------------------------------------------------------------------------------
    def _enqueue(self, r):
        self.prefills.append((r.arrival, self.seq, r))
        self.seq += 1
        self.prefills.sort(key=lambda e: (e[0], e[1]))       # arrival-time order

    def submit(self, rid, arrival, prompt_len, response_len, output_len):
        r = Request(rid, arrival, prompt_len, response_len, output_len, self.block)
        self.reqs[rid] = r
        self._enqueue(r)

    def _pages_needed(self, r):
        return -(-r.seq_len // PAGE)

    # ---- Algorithm 1 -----------------------------------------------------------------------------------------
    def schedule(self):
        """One iteration: returns (decodes, admitted prefills) as lists of requests, microbatch order."""
        decodes = list(self.decodes)
        if not self.prefills:
            self.deficit = 0
            self.last = (decodes, [])
            return self.last
        budget = self.tau - self.block * len(decodes) + self.deficit
        admitted = []
        rows = sum(min(self.block, r.seq_len - (r.prompt_len + r.cur_block * self.block)) for r in decodes)
        while self.prefills:
            p = self.prefills[0][2]
            idle = (len(decodes) + len(admitted) == 0)
            fits_memory = p.pages is not None or self._pages_needed(p) <= len(self.free_pages)
            if self.max_batch is not None and len(decodes) + len(admitted) >= self.max_batch:
                fits_memory = False
            if self.max_total_q is not None and rows + p.seq_len > self.max_total_q:
                fits_memory = False
            if (p.seq_len <= budget or idle) and fits_memory:
                rows += p.seq_len
                self.prefills.pop(0)
                if p.pages is None:
                    p.pages = [self.free_pages.pop() for _ in range(self._pages_needed(p))]
                admitted.append(p)
                budget -= p.seq_len
            else:
                break
        self.deficit = max(budget, 0)
        self.last = (decodes, admitted)
        return self.last

    # ---- after the model ran the microbatch --------------------------------------------------------------------
    def complete(self, block_done):
        """block_done[i] != 0: decode i of the last microbatch resolved its block in this iteration."""
        decodes, admitted = self.last
        assert len(block_done) == len(decodes)
        keep = []
        for r, done in zip(decodes, block_done):
            if not done:
                keep.append(r)
                continue
            r.cur_block += 1
            if r.cur_block >= r.nblocks:                      # retired: pages go back to the pool
                for pg in reversed(r.pages):
                    self.free_pages.append(pg)
                r.pages = None
                del self.reqs[r.rid]
            else:                                             # block boundary: cache refresh = re-prefill
                self._enqueue(r)
        self.decodes = keep + admitted                        # an admitted prefill decodes its current block next
        self.last = ([], [])

    # ---- batch metadata ----------------------------------------------------------------------------------------
    def metadata(self, width):
        """cu_q_lens, ctx_lens, block_table [R][width] (-1 padded), slot_mapping of the last scheduled microbatch."""
        decodes, admitted = self.last
        R = len(decodes) + len(admitted)
        q_lens, ctx, slots = [], [], []
        bt = np.full((R, width), -1, dtype=np.int32)
        for i, r in enumerate(decodes + admitted):
            is_decode = i < len(decodes)
            pages = np.asarray(r.pages, dtype=np.int64)
            bt[i, :len(pages)] = pages
            ctx.append(r.seq_len)
            if is_decode:
                first = r.prompt_len + r.cur_block * r.block
                pos = np.arange(first, min(first + r.block, r.seq_len))
            else:
                pos = np.arange(r.seq_len)
            q_lens.append(len(pos))
            slots.append(pages[pos // PAGE] * PAGE + pos % PAGE)
        cu = np.concatenate([[0], np.cumsum(q_lens)]).astype(np.int32)
        sm = np.concatenate(slots).astype(np.int32) if slots else np.zeros(0, np.int32)
        rid = np.asarray([r.rid for r in decodes + admitted], dtype=np.int64)
        return cu, np.asarray(ctx, dtype=np.int32), bt, sm, rid, len(decodes)
