// kv_host.h — host-side runtime of the D-instance KV pool: block allocator, request table,
// split-KV planner.  Pure C++17, no CUDA: everything here is integer bookkeeping (SURVEY §8(a)
// rows a1 and a6, and the work-list half of a4).  The paper prices none of this beyond noting
// that transfer cost depends on "block fragmentation and count" and that KV
// occupancy is a monitored signal.
#pragma once

#include <algorithm>
#include <cstdint>
#include <unordered_map>
#include <vector>

#include "../../include/kv_pool.h"

namespace kvp {

inline uint64_t splitmix64_next(uint64_t& state) {
  uint64_t z = (state += 0x9E3779B97F4A7C15ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// Free list of physical block ids.  pop() hands out ids from the back.
//   seed == 0 : initial order such that the first pops return 0, 1, 2, ...
//   seed != 0 : initial order is a Fisher-Yates permutation (fragmented pool).
// Freed blocks are pushed back and reused LIFO.
class BlockAllocator {
 public:
  void init(int64_t num_blocks, uint64_t seed) {
    total_ = num_blocks;
    free_.resize(static_cast<size_t>(num_blocks));
    for (int64_t i = 0; i < num_blocks; ++i) free_[static_cast<size_t>(i)] = static_cast<int32_t>(num_blocks - 1 - i);
    if (seed != 0) {
      uint64_t s = seed;
      for (int64_t i = num_blocks - 1; i > 0; --i) {
        uint64_t j = splitmix64_next(s) % static_cast<uint64_t>(i + 1);
        std::swap(free_[static_cast<size_t>(i)], free_[static_cast<size_t>(j)]);
      }
    }
    high_water_ = 0;
  }
  int64_t total() const { return total_; }
  int64_t free_count() const { return static_cast<int64_t>(free_.size()); }
  int64_t high_water() const { return high_water_; }
  int32_t pop() {
    int32_t b = free_.back();
    free_.pop_back();
    high_water_ = std::max(high_water_, total_ - free_count());
    return b;
  }
  void push(int32_t b) { free_.push_back(b); }
  void set_high_water(int64_t v) { high_water_ = v; }

 private:
  std::vector<int32_t> free_;
  int64_t total_ = 0, high_water_ = 0;
};

struct Request {
  int32_t slot = -1;    // row of the device block_table mirror
  int32_t len = 0;      // tokens stored (reserved)
  int32_t last_n = 0;   // size of the last reservation (for layer-sliced ingest)
  mutable uint64_t plan_mark = 0;  // duplicate detection in plan_decode / batch validation
  std::vector<int32_t> blocks;
};

// One split-KV work item: a run of logical blocks of one request, shared by all its KV heads.
// The kernel expands item i into num_kv_heads units (unit = i * Hkv + kv_head, heads fastest, so
// neighbouring warps stream neighbouring head tiles of the same physical blocks).
struct WorkItem {
  int32_t batch_idx;     // row of q / out
  int32_t slot;          // row of the device block_table
  int32_t blk_begin;     // first logical block
  int32_t n_blocks;
  int32_t n_tokens;      // valid tokens in this run (last block of a request may be partial)
  int32_t partial_base;  // first partial slot of this request, or -1: only chunk, writes `out`
  int32_t chunks;        // (n_chunks << 16) | chunk_idx; partial slot of (kv_head h, chunk c) =
                         //   partial_base + h * n_chunks + c
  int32_t last_blk;      // physical id of the request's LAST block (the fused decode step appends there
                         //   before the device block_table mirror has seen it)
};
static_assert(sizeof(WorkItem) == 32, "WorkItem is read by the kernel as two int4");

// One request that was split: its Hkv * G heads each merge n_chunks partials.
struct CombineEntry {
  int32_t batch_idx, partial_begin, n_chunks, pad;
};

struct DecodePlan {
  std::vector<WorkItem> items;
  std::vector<int32_t> item_span;   // index of the planned span (request / query tile) of each item
  std::vector<CombineEntry> combines;
  int32_t chunk_blocks = 0;
  int32_t n_partials = 0;
};

constexpr int32_t kMaxBlocksPerRequest = 131072;

class HostState {
 public:
  kv_pool_config_t cfg{};
  BlockAllocator alloc;
  std::unordered_map<int64_t, Request> reqs;
  std::vector<int32_t> free_slots;
  uint64_t epoch = 1;  // bumped whenever any request's blocks or length change

  static int32_t validate(const kv_pool_config_t& c) {
    if (c.num_layers < 1 || c.num_q_heads < 1 || c.num_kv_heads < 1) return KV_ERR_INVALID;
    if (c.head_dim != 64 && c.head_dim != 128) return KV_ERR_INVALID;
    if (c.block_size != 16) return KV_ERR_INVALID;
    if (c.kv_dtype != KV_DTYPE_BF16 && c.kv_dtype != KV_DTYPE_FP8_E4M3) return KV_ERR_INVALID;
    if (c.num_q_heads % c.num_kv_heads != 0 || c.num_q_heads / c.num_kv_heads > 8) return KV_ERR_INVALID;
    if (c.num_blocks < 1 || c.num_blocks > 0x7fffffffLL) return KV_ERR_INVALID;
    // <= 131072 blocks (2 Mi tokens) per request: lengths stay far inside int32, the (n_chunks, chunk) pair fits its
    // 16:16 packing, and one request's descriptor (48 B + 8 B per block for a transfer) fits an ingest blob
    if (c.max_requests < 1 || c.max_blocks_per_request < 1 || c.max_blocks_per_request > kMaxBlocksPerRequest) return KV_ERR_INVALID;
    if (static_cast<int64_t>(c.max_requests) * c.max_blocks_per_request > (1LL << 31)) return KV_ERR_INVALID;
    return KV_OK;
  }

  void init(const kv_pool_config_t& c) {
    cfg = c;
    alloc.init(c.num_blocks, c.alloc_seed);
    free_slots.resize(static_cast<size_t>(c.max_requests));
    for (int32_t i = 0; i < c.max_requests; ++i) free_slots[static_cast<size_t>(i)] = c.max_requests - 1 - i;
  }

  int32_t blocks_for(int64_t tokens) const {
    return static_cast<int32_t>((tokens + cfg.block_size - 1) / cfg.block_size);
  }

  // a1.  Atomic over the batch: validate everything, then mutate.
  int32_t reserve(int32_t n_req, const int64_t* ids, const int32_t* n_tokens) {
    if (n_req < 0 || (n_req > 0 && (!ids || !n_tokens))) return KV_ERR_INVALID;
    const uint64_t stamp = ++plan_stamp_;
    fresh_.clear();
    int64_t need_blocks = 0;
    for (int32_t i = 0; i < n_req; ++i) {
      if (n_tokens[i] < 0) return KV_ERR_INVALID;
      auto it = reqs.find(ids[i]);
      int64_t len = 0;
      if (it == reqs.end()) {
        fresh_.push_back(ids[i]);
      } else {
        if (it->second.plan_mark == stamp) return KV_ERR_INVALID;  // duplicate id
        it->second.plan_mark = stamp;
        len = it->second.len;
      }
      int64_t new_len = len + n_tokens[i];
      if (new_len > static_cast<int64_t>(cfg.max_blocks_per_request) * cfg.block_size) return KV_ERR_TOO_LONG;
      need_blocks += blocks_for(new_len) - blocks_for(len);
    }
    if (fresh_.size() > 1) {  // duplicates among the ids that are not live yet
      std::sort(fresh_.begin(), fresh_.end());
      if (std::adjacent_find(fresh_.begin(), fresh_.end()) != fresh_.end()) return KV_ERR_INVALID;
    }
    if (fresh_.size() > free_slots.size()) return KV_ERR_TOO_MANY_REQUESTS;
    if (need_blocks > alloc.free_count()) return KV_ERR_NO_BLOCKS;
    undo_.clear();
    undo_high_water_ = alloc.high_water();
    for (int32_t i = 0; i < n_req; ++i) {
      auto it = reqs.find(ids[i]);
      const bool created = it == reqs.end();
      if (created) {
        Request r;
        r.slot = free_slots.back();
        free_slots.pop_back();
        it = reqs.emplace(ids[i], std::move(r)).first;
      }
      Request& r = it->second;
      undo_.push_back({ids[i], r.last_n, n_tokens[i], created});
      int32_t want = blocks_for(static_cast<int64_t>(r.len) + n_tokens[i]);
      while (static_cast<int32_t>(r.blocks.size()) < want) r.blocks.push_back(alloc.pop());
      r.len += n_tokens[i];
      r.last_n = n_tokens[i];
    }
    ++epoch;
    return KV_OK;
  }

  // Undo the LAST successful reserve() exactly (a call that reserved and then could not launch must leave the
  // pool as it found it): blocks go back in reverse order of their pops, so the free list, the slot list and the
  // high-water mark are what they were; requests the reservation created are dropped.
  void rollback_last_reserve() {
    for (auto u = undo_.rbegin(); u != undo_.rend(); ++u) {
      auto it = reqs.find(u->id);
      Request& r = it->second;
      r.len -= u->n_tokens;
      r.last_n = u->prev_last_n;
      const int32_t want = blocks_for(r.len);
      while (static_cast<int32_t>(r.blocks.size()) > want) { alloc.push(r.blocks.back()); r.blocks.pop_back(); }
      if (u->created) { free_slots.push_back(r.slot); reqs.erase(it); }
    }
    alloc.set_high_water(undo_high_water_);
    undo_.clear();
    ++epoch;
  }

  // a6.  Atomic: unknown or duplicate id => nothing freed.
  int32_t release(int32_t n_req, const int64_t* ids) {
    if (n_req < 0 || (n_req > 0 && !ids)) return KV_ERR_INVALID;
    const uint64_t stamp = ++plan_stamp_;
    for (int32_t i = 0; i < n_req; ++i) {
      auto it = reqs.find(ids[i]);
      if (it == reqs.end()) return KV_ERR_UNKNOWN_REQUEST;
      if (it->second.plan_mark == stamp) return KV_ERR_INVALID;
      it->second.plan_mark = stamp;
    }
    for (int32_t i = 0; i < n_req; ++i) {
      auto it = reqs.find(ids[i]);
      Request& r = it->second;
      for (auto b = r.blocks.rbegin(); b != r.blocks.rend(); ++b) alloc.push(*b);
      free_slots.push_back(r.slot);
      reqs.erase(it);
    }
    ++epoch;
    return KV_OK;
  }

  // Every id live, none repeated (continuation ingest, host-buffer attention).  Optionally requires
  // each request's last reservation to equal n_tokens[i].
  int32_t check_batch(int32_t n_req, const int64_t* ids, const int32_t* last_n) const {
    const uint64_t stamp = ++plan_stamp_;
    for (int32_t i = 0; i < n_req; ++i) {
      auto it = reqs.find(ids[i]);
      if (it == reqs.end()) return KV_ERR_UNKNOWN_REQUEST;
      if (it->second.plan_mark == stamp) return KV_ERR_INVALID;
      it->second.plan_mark = stamp;
      if (last_n && it->second.last_n != last_n[i]) return KV_ERR_INVALID;
    }
    return KV_OK;
  }

  // Work-list half of a4: decode.  One span per request (row = batch index), all its blocks.
  int32_t plan_decode(int32_t batch, const int64_t* ids, int32_t slots, int32_t items_per_slot,
                      int32_t min_chunk_blocks, int32_t max_partials, DecodePlan* plan) const {
    if (batch < 1 || !ids || batch > cfg.max_requests) return KV_ERR_INVALID;
    spans_.resize(static_cast<size_t>(batch));
    const uint64_t stamp = ++plan_stamp_;
    for (int32_t i = 0; i < batch; ++i) {
      auto it = reqs.find(ids[i]);
      if (it == reqs.end()) return KV_ERR_UNKNOWN_REQUEST;
      const Request& r = it->second;
      if (r.len < 1 || r.plan_mark == stamp) return KV_ERR_INVALID;  // empty context (A11) / duplicate id
      r.plan_mark = stamp;
      spans_[static_cast<size_t>(i)] = {i, r.slot, blocks_for(r.len), r.len, r.blocks.back()};
    }
    return plan_spans(slots, items_per_slot, min_chunk_blocks, max_partials, plan);
  }

  // Work-list half of the variable-q-length call: request i's
  // LAST q_lens[i] tokens are query tokens (a decode row has q_lens[i] = 1, an in-place prefill row
  // q_lens[i] = its prompt length).  The kernel packs (query token, head) pairs into its 8 MMA
  // columns, so the unit of planning is a QUERY TILE of 8 / G consecutive query tokens: one span per
  // tile, covering the blocks that hold tokens 0 .. position of the tile's last query token (causal).
  // plan->items[k].batch_idx = first row of the tile in q / out; tiles[k] = {pos0, n_qtok} for the
  // same k (pos0 = absolute position of the tile's first query token).
  struct QueryTile { int32_t pos0, n_qtok; };
  int32_t plan_varq(int32_t batch, const int64_t* ids, const int32_t* q_lens, int32_t slots, int32_t items_per_slot,
                    int32_t min_chunk_blocks, int32_t max_partials, DecodePlan* plan,
                    std::vector<QueryTile>* tiles) const {
    if (batch < 1 || !ids || !q_lens || batch > cfg.max_requests) return KV_ERR_INVALID;
    const int32_t G = cfg.num_q_heads / cfg.num_kv_heads;
    const int32_t tpt = std::max(1, 8 / G);   // query tokens per tile
    spans_.clear();
    span_tiles_.clear();
    const uint64_t stamp = ++plan_stamp_;
    int64_t row = 0;
    for (int32_t i = 0; i < batch; ++i) {
      auto it = reqs.find(ids[i]);
      if (it == reqs.end()) return KV_ERR_UNKNOWN_REQUEST;
      const Request& r = it->second;
      if (q_lens[i] < 1 || q_lens[i] > r.len || r.plan_mark == stamp) return KV_ERR_INVALID;
      r.plan_mark = stamp;
      const int32_t p0 = r.len - q_lens[i];
      for (int32_t k = 0; k < q_lens[i]; k += tpt) {
        const int32_t nq = std::min(tpt, q_lens[i] - k);
        const int32_t visible = p0 + k + nq;                      // tokens 0 .. position of the tile's last query
        if (row + k > 0x7fffffff) return KV_ERR_TOO_LONG;
        spans_.push_back({static_cast<int32_t>(row + k), r.slot, blocks_for(visible), visible, r.blocks.back()});
        span_tiles_.push_back({p0 + k, nq});
      }
      row += q_lens[i];
    }
    int32_t rc = plan_spans(slots, items_per_slot, min_chunk_blocks, max_partials, plan);
    if (rc != KV_OK) return rc;
    tiles->resize(plan->items.size());
    for (size_t k = 0; k < plan->items.size(); ++k) (*tiles)[k] = span_tiles_[static_cast<size_t>(plan->item_span[k])];
    return KV_OK;
  }

 private:
  // One independently planned run of blocks [0, nb) with n_tokens valid tokens: a request (decode)
  // or a query tile (variable-q).  `row` lands in WorkItem::batch_idx.
  struct Span { int32_t row, slot, nb, n_tokens, last_blk; };

  // `slots` = resident warps the main kernel will run (one work unit at a time each; an item expands
  // to num_kv_heads units).  Chunk sizes follow guided self-scheduling: spans are taken longest
  // first and each chunk is sized to the work still unassigned,
  //     c = max(min_chunk_blocks, remaining_tiles / (items_per_slot * slots))   blocks,
  // so the list starts with few large units (few unit switches, few partials) and ends with small
  // ones (the warps, which claim units dynamically in list order, all finish within one small
  // unit of each other).  A span whose remainder is <= 1.25 c is not split further.
  // Cost matters (a 7B-MHA decode step is ~0.2 ms of GPU time): two passes over the spans, counting sorts.
  int32_t plan_spans(int32_t slots, int32_t items_per_slot, int32_t min_chunk_blocks, int32_t max_partials,
                     DecodePlan* plan) const {
    const int32_t n_spans = static_cast<int32_t>(spans_.size());
    int64_t total_blocks = 0;
    int32_t longest = 0;
    for (const Span& sp : spans_) {
      total_blocks += sp.nb;
      longest = std::max(longest, sp.nb);
    }
    // longest span first (stable counting sort on the block count)
    order_.resize(static_cast<size_t>(n_spans));
    count_.assign(static_cast<size_t>(longest) + 2, 0);
    for (const Span& sp : spans_) ++count_[static_cast<size_t>(longest - sp.nb) + 1];
    for (size_t k = 1; k < count_.size(); ++k) count_[k] += count_[k - 1];
    for (int32_t i = 0; i < n_spans; ++i)
      order_[static_cast<size_t>(count_[static_cast<size_t>(longest - spans_[static_cast<size_t>(i)].nb)]++)] = i;

    const int64_t Hkv = cfg.num_kv_heads;
    const int64_t denom = std::max<int64_t>(1, static_cast<int64_t>(slots) * items_per_slot);
    int64_t floor_blocks = std::max<int32_t>(1, min_chunk_blocks);
    int32_t max_nb = 0, next_partial = 0;
    for (;;) {  // raise the smallest chunk until the partials fit the workspace
      unsorted_.clear();
      unsorted_span_.clear();
      plan->combines.clear();
      next_partial = 0;
      max_nb = 0;
      int64_t remaining = total_blocks * Hkv;  // tiles not yet assigned
      bool overflow = false;
      for (int32_t oi = 0; oi < n_spans && !overflow; ++oi) {
        const int32_t i = order_[static_cast<size_t>(oi)];
        const Span& sp = spans_[static_cast<size_t>(i)];
        const size_t first = unsorted_.size();
        int32_t pos = 0;
        while (pos < sp.nb) {
          const int64_t c = std::max<int64_t>(floor_blocks, remaining / denom);
          const int32_t rem = sp.nb - pos;
          const int32_t take = rem <= c + c / 4 ? rem : static_cast<int32_t>(c);
          WorkItem w;
          w.batch_idx = sp.row;
          w.slot = sp.slot;
          w.blk_begin = pos;
          w.n_blocks = take;
          w.n_tokens = std::min(sp.n_tokens - pos * cfg.block_size, take * cfg.block_size);
          w.partial_base = -1;
          w.chunks = 0;
          w.last_blk = sp.last_blk;
          unsorted_.push_back(w);
          unsorted_span_.push_back(i);
          max_nb = std::max(max_nb, take);
          pos += take;
          remaining -= take * Hkv;
        }
        const int32_t nc = static_cast<int32_t>(unsorted_.size() - first);
        if (nc > 0xffff) return KV_ERR_TOO_LONG;   // (n_chunks, chunk_idx) are packed 16:16
        if (nc > 1) {
          if (static_cast<int64_t>(next_partial) + static_cast<int64_t>(nc) * Hkv > max_partials) { overflow = true; break; }
          plan->combines.push_back({sp.row, next_partial, nc, 0});
          for (int32_t c = 0; c < nc; ++c) unsorted_[first + static_cast<size_t>(c)].partial_base = next_partial;
          next_partial += nc * static_cast<int32_t>(Hkv);
        }
        for (int32_t c = 0; c < nc; ++c) unsorted_[first + static_cast<size_t>(c)].chunks = (nc << 16) | c;
      }
      if (!overflow) break;
      if (floor_blocks > longest) return KV_ERR_TOO_LONG;   // even unsplit spans do not fit: cannot happen (no partials then)
      floor_blocks *= 2;
    }
    {  // largest chunk this plan may contain (first chunk target, plus the no-split allowance)
      const int64_t c0 = std::max<int64_t>(floor_blocks, total_blocks * Hkv / denom);
      plan->chunk_blocks = static_cast<int32_t>(std::min<int64_t>(c0 + c0 / 4, 0x7fffffff));
    }
    plan->n_partials = next_partial;
    // largest units first, stable: counting sort on n_blocks
    count_.assign(static_cast<size_t>(max_nb) + 2, 0);
    for (const WorkItem& w : unsorted_) ++count_[static_cast<size_t>(max_nb - w.n_blocks) + 1];
    for (size_t k = 1; k < count_.size(); ++k) count_[k] += count_[k - 1];
    plan->items.resize(unsorted_.size());
    plan->item_span.resize(unsorted_.size());
    for (size_t k = 0; k < unsorted_.size(); ++k) {
      const int32_t dst = count_[static_cast<size_t>(max_nb - unsorted_[k].n_blocks)]++;
      plan->items[static_cast<size_t>(dst)] = unsorted_[k];
      plan->item_span[static_cast<size_t>(dst)] = unsorted_span_[k];
    }
    return KV_OK;
  }

  mutable std::vector<Span> spans_;
  mutable std::vector<QueryTile> span_tiles_;
  mutable std::vector<int32_t> unsorted_span_;
  mutable std::vector<WorkItem> unsorted_;
  mutable std::vector<int32_t> count_, order_;
  std::vector<int64_t> fresh_;
  struct Undo { int64_t id; int32_t prev_last_n, n_tokens; bool created; };
  std::vector<Undo> undo_;
  int64_t undo_high_water_ = 0;
  mutable uint64_t plan_stamp_ = 0;
};

}  // namespace kvp
