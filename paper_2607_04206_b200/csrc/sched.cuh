// sched.cuh -- the worker-level deficit token-budget scheduler (Algorithm 1) and the builder of the
// batch metadata the kernels consume (cu_q_lens / ctx_lens / block_table / slot_mapping).
// Plain host C++ (integer logic, no device work); exported through the C ABI of include/sangam.h as sangam_sched_*.
// It shares no code with oracle/sched_oracle.py.
//
// Algorithm 1, as implemented by sangam_sched_next (line numbers of the listing at):
//    1-4   no waiting prefill: deficit <- 0, the microbatch is the in-flight decodes (decode-only iteration)
//    5     budget <- tau - Tokens(decodes) + deficit           Tokens(decode) = one block, Tokens(prefill) = prompt + response
//    6     microbatch <- decodes                               decodes are never displaced
//    7-16  while a prefill waits: p <- head of the queue (arrival-time order);
//          idle <- microbatch empty; admit p if Tokens(p) <= budget or idle (liveness), budget -= Tokens(p);
//          otherwise stop: the first prefill that does not fit ends the scan, prefills are never split
//    17    deficit <- max(budget, 0)
// Readings beyond the listing (S20-S22): equal arrival times keep submission order; a head prefill whose KV
// pages do not fit the free pool, or that would exceed the ctx capacities (max_batch, max_total_q), "does not fit" and
// stops the scan without spending budget, also under the idle rule; a request's pages are taken at its first admission
// and returned when its last block resolves.
#pragma once
#include <stdint.h>

#include <algorithm>
#include <new>
#include <unordered_map>
#include <vector>

#include "../../include/sangam.h"
#include "common.cuh"

struct SchedReq {
    int64_t rid;
    double arrival;
    int32_t prompt_len, response_len, nblocks, cur_block;
    std::vector<int32_t> pages;      // empty until the first admission
    bool live;
};
struct SchedWaiting {
    double arrival;
    uint64_t seq;
    int32_t slot;
};

struct sangam_sched {
    sangam_sched_config cfg;
    int64_t deficit;
    uint64_t seq;
    std::vector<SchedReq> reqs;
    std::vector<int32_t> free_slots;
    std::unordered_map<int64_t, int32_t> by_id;
    std::vector<int32_t> decodes;            // request slots, in the order they became decodes
    std::vector<SchedWaiting> prefills;      // sorted by (arrival, seq)
    std::vector<int32_t> free_pages;         // stack: back() is the next page handed out (0, 1, 2, ... from a fresh pool)
    std::vector<int32_t> last_decodes, last_prefills;
    bool scheduled;
};

static inline int32_t sched_pages_needed(const SchedReq& r) { return (r.prompt_len + r.response_len + SANGAM_PAGE - 1) / SANGAM_PAGE; }
static inline int32_t sched_seq_len(const SchedReq& r) { return r.prompt_len + r.response_len; }

static inline void sched_enqueue(sangam_sched* s, int32_t slot) {
    SchedWaiting w{s->reqs[slot].arrival, s->seq++, slot};
    auto pos = std::upper_bound(s->prefills.begin(), s->prefills.end(), w, [](const SchedWaiting& a, const SchedWaiting& b) {
        return a.arrival < b.arrival || (a.arrival == b.arrival && a.seq < b.seq);
    });
    s->prefills.insert(pos, w);
}

extern "C" int sangam_sched_create(const sangam_sched_config* cfg, sangam_sched** out) {
    if (!cfg || !out) return SANGAM_ERR_INVALID_ARG;
    *out = nullptr;
    if (cfg->page_size != SANGAM_PAGE) return SANGAM_ERR_UNSUPPORTED;
    if (cfg->tau <= 0 || cfg->block <= 0 || cfg->num_pages <= 0 || cfg->max_batch <= 0 || cfg->max_total_q <= 0 || cfg->max_pages_per_req <= 0)
        return SANGAM_ERR_INVALID_ARG;
    sangam_sched* s = new (std::nothrow) sangam_sched();
    if (!s) return SANGAM_ERR_WORKSPACE;
    s->cfg = *cfg;
    s->deficit = 0; s->seq = 0; s->scheduled = false;
    s->free_pages.resize(cfg->num_pages);
    for (int32_t i = 0; i < cfg->num_pages; ++i) s->free_pages[i] = cfg->num_pages - 1 - i;
    *out = s;
    return SANGAM_OK;
}

extern "C" int sangam_sched_destroy(sangam_sched* s) {
    if (!s) return SANGAM_ERR_INVALID_ARG;
    delete s;
    return SANGAM_OK;
}

extern "C" int sangam_sched_submit(sangam_sched* s, int64_t req_id, double arrival_time, int32_t prompt_len, int32_t response_len,
                                   int32_t output_len) {
    if (!s || prompt_len < 0 || response_len <= 0 || output_len <= 0) return SANGAM_ERR_INVALID_ARG;
    if (s->by_id.count(req_id)) return SANGAM_ERR_INVALID_ARG;
    SchedReq r;
    r.rid = req_id; r.arrival = arrival_time; r.prompt_len = prompt_len; r.response_len = response_len;
    const int32_t out_len = output_len < response_len ? output_len : response_len;
    r.nblocks = (out_len + s->cfg.block - 1) / s->cfg.block;          // blocks past the committed EOS are never denoised
    if (r.nblocks < 1) r.nblocks = 1;
    r.cur_block = 0; r.live = true;
    // a request that can never be scheduled is refused here rather than blocking the queue for ever
    if (sched_pages_needed(r) > s->cfg.max_pages_per_req || sched_pages_needed(r) > s->cfg.num_pages || sched_seq_len(r) > s->cfg.max_total_q)
        return SANGAM_ERR_WORKSPACE;
    int32_t slot;
    if (!s->free_slots.empty()) { slot = s->free_slots.back(); s->free_slots.pop_back(); s->reqs[slot] = r; }
    else { slot = (int32_t)s->reqs.size(); s->reqs.push_back(r); }
    s->by_id[req_id] = slot;
    sched_enqueue(s, slot);
    return SANGAM_OK;
}

extern "C" int sangam_sched_next(sangam_sched* s, sangam_batch* out) {
    if (!s || !out) return SANGAM_ERR_INVALID_ARG;
    const sangam_sched_config& c = s->cfg;
    s->last_decodes = s->decodes;
    s->last_prefills.clear();
    int64_t rows = 0;
    for (int32_t slot : s->decodes) {
        const SchedReq& r = s->reqs[slot];
        const int32_t first = r.prompt_len + r.cur_block * c.block;
        rows += std::min(c.block, sched_seq_len(r) - first);
    }
    if (s->prefills.empty()) {
        s->deficit = 0;                                               // decode-only iteration (lines 1-4)
    } else {
        int64_t budget = (int64_t)c.tau - (int64_t)c.block * (int64_t)s->decodes.size() + s->deficit;
        while (!s->prefills.empty()) {
            const int32_t slot = s->prefills.front().slot;
            SchedReq& p = s->reqs[slot];
            const bool idle = s->decodes.empty() && s->last_prefills.empty();
            const int64_t tokens = sched_seq_len(p);
            const bool has_room = (int64_t)(s->decodes.size() + s->last_prefills.size()) < c.max_batch && rows + tokens <= c.max_total_q &&
                                  (!p.pages.empty() || sched_pages_needed(p) <= (int32_t)s->free_pages.size());
            if ((tokens <= budget || idle) && has_room) {
                s->prefills.erase(s->prefills.begin());
                if (p.pages.empty()) {
                    const int32_t n = sched_pages_needed(p);
                    p.pages.resize(n);
                    for (int32_t i = 0; i < n; ++i) { p.pages[i] = s->free_pages.back(); s->free_pages.pop_back(); }
                }
                s->last_prefills.push_back(slot);
                budget -= tokens;
                rows += tokens;
            } else {
                break;                                                // p waits; prefills cannot be split
            }
        }
        s->deficit = budget > 0 ? budget : 0;
    }
    s->scheduled = true;
    // ---- batch metadata: decodes first, then the admitted prefills
    const int32_t nd = (int32_t)s->last_decodes.size(), np = (int32_t)s->last_prefills.size(), R = nd + np;
    out->batch = R; out->num_decodes = nd; out->deficit = s->deficit;
    int32_t q = 0;
    if (out->cu_q_lens) out->cu_q_lens[0] = 0;
    for (int32_t i = 0; i < R; ++i) {
        const SchedReq& r = s->reqs[i < nd ? s->last_decodes[i] : s->last_prefills[i - nd]];
        const int32_t first = i < nd ? r.prompt_len + r.cur_block * c.block : 0;
        const int32_t last = i < nd ? std::min(first + c.block, sched_seq_len(r)) : sched_seq_len(r);
        if (out->req_ids) out->req_ids[i] = r.rid;
        if (out->ctx_lens) out->ctx_lens[i] = sched_seq_len(r);
        if (out->block_table) {
            int32_t* row = out->block_table + (int64_t)i * c.max_pages_per_req;
            const int32_t n = (int32_t)r.pages.size();
            for (int32_t j = 0; j < c.max_pages_per_req; ++j) row[j] = j < n ? r.pages[j] : -1;
        }
        if (out->slot_mapping)
            for (int32_t pos = first; pos < last; ++pos) out->slot_mapping[q + pos - first] = r.pages[pos / SANGAM_PAGE] * SANGAM_PAGE + pos % SANGAM_PAGE;
        q += last - first;
        if (out->cu_q_lens) out->cu_q_lens[i + 1] = q;
    }
    out->total_q = q;
    out->num_new_tokens = q;                                         // every query row's K/V is (re)written this iteration
    return SANGAM_OK;
}

extern "C" int sangam_sched_complete(sangam_sched* s, const int32_t* block_done, int32_t n) {
    if (!s || n < 0 || (n > 0 && !block_done)) return SANGAM_ERR_INVALID_ARG;
    if (!s->scheduled || n != (int32_t)s->last_decodes.size()) return SANGAM_ERR_INVALID_ARG;
    std::vector<int32_t> keep;
    for (int32_t i = 0; i < n; ++i) {
        const int32_t slot = s->last_decodes[i];
        SchedReq& r = s->reqs[slot];
        if (!block_done[i]) { keep.push_back(slot); continue; }
        if (++r.cur_block >= r.nblocks) {                             // retired: pages return to the pool (last taken, first back)
            for (auto it = r.pages.rbegin(); it != r.pages.rend(); ++it) s->free_pages.push_back(*it);
            r.pages.clear(); r.live = false;
            s->by_id.erase(r.rid);
            s->free_slots.push_back(slot);
        } else {
            sched_enqueue(s, slot);                                   // block boundary: cache refresh = re-prefill, original arrival time
        }
    }
    keep.insert(keep.end(), s->last_prefills.begin(), s->last_prefills.end());     // an admitted prefill decodes next
    s->decodes.swap(keep);
    s->last_decodes.clear(); s->last_prefills.clear();
    s->scheduled = false;
    return SANGAM_OK;
}

extern "C" int64_t sangam_sched_query(const sangam_sched* s, int32_t what) {
    if (!s) return -1;
    switch (what) {
        case SANGAM_SCHED_DEFICIT: return s->deficit;
        case SANGAM_SCHED_WAITING: return (int64_t)s->prefills.size();
        case SANGAM_SCHED_IN_FLIGHT: return (int64_t)s->decodes.size();
        case SANGAM_SCHED_FREE_PAGES: return (int64_t)s->free_pages.size();
        case SANGAM_SCHED_LIVE_REQUESTS: return (int64_t)s->by_id.size();
        default: return -1;
    }
}
