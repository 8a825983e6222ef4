// ks_sched.cu — the serving scheduler (host logic) and the closed simulation loop over the GPU path.
// SURVEY.md §8(f) NEXT-4; PAPER.md:241-249 (scheduler, mixed-step pricing), :231 (layer-homogeneous
// step body), :159 (a step completes at now + t_step).  Rules: DESIGN.md Q18.
//
// The scheduler is plain C++ with no device code.  ks_sim_run drives many of them in lock step and
// prices every iteration's batches with ONE pass of the library's own GPU path: rows are packed into
// one pinned arena, run through ks_run_steps (device space), and the step times land in the same arena.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <chrono>
#include <cstring>
#include <deque>
#include <limits>
#include <list>
#include <new>
#include <unordered_map>
#include <vector>

#include "ks_internal.h"

struct ks_sched {
  ks_sched_config cfg{};
  // per request, insertion order
  std::vector<double> arrival, first_token, finish;
  std::vector<int32_t> prompt, max_new, n_tok, computed, generated, blocks, n_preempt;
  std::vector<int32_t> order;          // FCFS order: (arrival, insertion index)
  size_t next_pos = 0;                 // first entry of `order` that has not arrived yet
  bool started = false;
  std::deque<int32_t> waiting;
  std::vector<int32_t> running;
  // the batch being executed
  std::vector<int32_t> b_req, b_new, b_hist;
  bool pending = false;
  int32_t free_blocks = 0;             // blocks holding nothing (cached blocks nobody references are in `lru`)
  int64_t n_steps = 0, tokens = 0, preemptions = 0;
  int32_t n_finished = 0;

  // prefix cache (Q19).  Key of full block j of prefix content p: p << 32 | j.
  struct GpuBlock {
    int32_t ref = 0;
    std::list<uint64_t>::iterator pos;   // position in `lru` while ref == 0
  };
  std::vector<int32_t> prefix_id, prefix_len, registered, cached_tokens;
  std::vector<std::vector<uint64_t>> held;                 // keys a request holds a reference on
  std::unordered_map<uint64_t, GpuBlock> gpu;              // GPU tier
  std::list<uint64_t> lru;                                 // unreferenced cached blocks, least recently released first
  std::list<uint64_t> disk_order;                          // disk tier, least recently used first
  std::unordered_map<uint64_t, std::list<uint64_t>::iterator> disk;
  int64_t gpu_hits = 0, disk_hits = 0, evictions = 0;
  std::vector<uint64_t> hit_keys;                          // scratch of the admission lookup
  std::vector<uint8_t> hit_on_disk;

  int32_t blocks_for(int64_t tokens_) const { return (int32_t)((tokens_ + cfg.block_size - 1) / cfg.block_size); }
  int32_t avail() const { return free_blocks + (int32_t)lru.size(); }
  static uint64_t key_of(int32_t p, int32_t j) { return ((uint64_t)(uint32_t)p << 32) | (uint32_t)j; }

  // k <= avail() blocks for a request: free ones first, then the least recently released cached ones
  void alloc(int32_t k) {
    const int32_t from_free = std::min(k, free_blocks);
    free_blocks -= from_free;
    for (k -= from_free; k > 0; --k) {
      gpu.erase(lru.front());
      lru.pop_front();
      ++evictions;
    }
  }
  // request r gives everything back: private blocks become free, shared ones lose a reference
  void release(int32_t r) {
    free_blocks += blocks[r] - (int32_t)held[r].size();
    for (uint64_t key : held[r]) {
      GpuBlock& g = gpu[key];
      if (--g.ref == 0) g.pos = lru.insert(lru.end(), key);
    }
    held[r].clear();
    blocks[r] = 0;
    registered[r] = 0;
  }
  void disk_put(uint64_t key) {
    if (cfg.disk_blocks <= 0) return;
    auto it = disk.find(key);
    if (it != disk.end()) {
      disk_order.splice(disk_order.end(), disk_order, it->second);
      return;
    }
    disk[key] = disk_order.insert(disk_order.end(), key);
    if ((int64_t)disk_order.size() > cfg.disk_blocks) {
      disk.erase(disk_order.front());
      disk_order.pop_front();
    }
  }
  // leading run of r's prefix blocks found in the GPU tier, else the disk tier; one token is always left
  void lookup(int32_t r) {
    hit_keys.clear();
    hit_on_disk.clear();
    if (!cfg.enable_prefix_cache || prefix_id[r] < 0) return;
    const int32_t limit = std::min(prefix_len[r] / cfg.block_size, (n_tok[r] - 1) / cfg.block_size);
    for (int32_t j = 0; j < limit; ++j) {
      const uint64_t key = key_of(prefix_id[r], j);
      if (gpu.count(key)) hit_on_disk.push_back(0);
      else if (disk.count(key)) hit_on_disk.push_back(1);
      else break;
      hit_keys.push_back(key);
    }
  }
};

namespace {

void sched_start(ks_sched* s) {
  const int n = (int)s->arrival.size();
  s->order.resize(n);
  for (int i = 0; i < n; ++i) s->order[i] = i;
  std::stable_sort(s->order.begin(), s->order.end(),
                   [s](int32_t a, int32_t b) { return s->arrival[a] < s->arrival[b]; });
  s->started = true;
}

// The token-budget loop.  Fills s->b_* with the batch of the step that starts at `now`.
void sched_form_batch(ks_sched* s, double now) {
  if (!s->started) sched_start(s);
  while (s->next_pos < s->order.size() && s->arrival[s->order[s->next_pos]] <= now) s->waiting.push_back(s->order[s->next_pos++]);
  s->b_req.clear(); s->b_new.clear(); s->b_hist.clear();
  int32_t budget = s->cfg.max_num_batched_tokens;
  bool preempted = false;
  auto take = [s, &budget](int32_t r, int32_t n_new, int32_t need) {
    s->alloc(need);
    s->blocks[r] += need;
    s->b_req.push_back(r); s->b_new.push_back(n_new); s->b_hist.push_back(s->computed[r]);
    budget -= n_new;
  };
  // running requests first, in queue order
  for (size_t i = 0; i < s->running.size() && budget > 0;) {
    const int32_t r = s->running[i];
    const int32_t n_new = std::min(s->n_tok[r] - s->computed[r], budget);
    const int32_t need = s->blocks_for((int64_t)s->computed[r] + n_new) - s->blocks[r];
    bool self = false;
    while (need > s->avail()) {            // KV pressure: the back of the running queue is recomputed later
      const int32_t v = s->running.back();
      s->running.pop_back();
      s->release(v);
      s->computed[v] = 0;
      ++s->n_preempt[v];
      ++s->preemptions;
      s->waiting.push_front(v);
      preempted = true;
      if (v == r) { self = true; break; }
    }
    if (self) break;
    take(r, n_new, need);
    ++i;
  }
  // FCFS admission (a partial chunk of a prompt is admitted with the budget that is left)
  if (!preempted) {
    while (!s->waiting.empty() && budget > 0 && (int32_t)s->running.size() < s->cfg.max_num_seqs) {
      const int32_t r = s->waiting.front();
      // prefix-cache-aware admission: cached leading blocks are referenced (GPU tier) or loaded (disk tier)
      // instead of recomputed; a waiting request always starts from computed == 0
      s->lookup(r);
      const int32_t n_hit = (int32_t)s->hit_keys.size();
      const int32_t hit = n_hit * s->cfg.block_size;
      const int32_t n_new = std::min(s->n_tok[r] - hit, budget);
      const int32_t need = s->blocks_for((int64_t)hit + n_new) - n_hit;
      int32_t taken = need;                 // blocks that leave the allocatable pool
      for (int32_t j = 0; j < n_hit; ++j) taken += s->hit_on_disk[j] ? 1 : (s->gpu[s->hit_keys[j]].ref == 0 ? 1 : 0);
      if (taken > s->avail()) break;
      for (int32_t j = 0; j < n_hit; ++j) {          // reference the GPU hits first: they must not be evicted below
        if (s->hit_on_disk[j]) continue;
        ks_sched::GpuBlock& g = s->gpu[s->hit_keys[j]];
        if (g.ref++ == 0) s->lru.erase(g.pos);
        ++s->gpu_hits;
      }
      for (int32_t j = 0; j < n_hit; ++j) {
        if (!s->hit_on_disk[j]) continue;
        s->alloc(1);
        s->gpu[s->hit_keys[j]].ref = 1;
        s->disk_put(s->hit_keys[j]);
        ++s->disk_hits;
      }
      s->held[r].assign(s->hit_keys.begin(), s->hit_keys.end());
      s->registered[r] = n_hit;
      s->blocks[r] = n_hit;
      s->computed[r] = hit;
      s->cached_tokens[r] += hit;
      s->waiting.pop_front();
      s->running.push_back(r);
      take(r, n_new, need);
    }
  }
  s->pending = !s->b_req.empty();
}

double sched_next_arrival(const ks_sched* s) {
  return s->next_pos < s->order.size() ? s->arrival[s->order[s->next_pos]] : std::numeric_limits<double>::infinity();
}

void sched_commit(ks_sched* s, double t_end) {
  for (size_t k = 0; k < s->b_req.size(); ++k) {
    const int32_t r = s->b_req[k];
    s->computed[r] += s->b_new[k];
    s->tokens += s->b_new[k];
    if (s->cfg.enable_prefix_cache && s->prefix_id[r] >= 0) {
      // full prefix blocks whose KV now exists go to the cache (one of r's private blocks becomes the shared
      // copy; if the key is already cached r keeps a private duplicate) and, written through, to the disk tier
      const int32_t full = std::min(s->computed[r], s->prefix_len[r]) / s->cfg.block_size;
      for (int32_t j = s->registered[r]; j < full; ++j) {
        const uint64_t key = ks_sched::key_of(s->prefix_id[r], j);
        if (!s->gpu.count(key)) {
          s->gpu[key].ref = 1;
          s->held[r].push_back(key);
        }
        s->disk_put(key);
      }
      s->registered[r] = std::max(s->registered[r], full);
    }
    if (s->computed[r] != s->n_tok[r]) continue;
    if (++s->generated[r] == 1) s->first_token[r] = t_end;
    if (s->generated[r] == s->max_new[r]) {
      s->finish[r] = t_end;
      s->release(r);
      s->running.erase(std::find(s->running.begin(), s->running.end(), r));
      ++s->n_finished;
    } else {
      ++s->n_tok[r];
    }
  }
  if (!s->b_req.empty()) ++s->n_steps;
  s->b_req.clear(); s->b_new.clear(); s->b_hist.clear();
  s->pending = false;
}

bool sched_done(const ks_sched* s) { return s->n_finished == (int32_t)s->arrival.size(); }

}  // namespace

extern "C" {

ks_status ks_sched_create(ks_sched** out, const ks_sched_config* cfg) {
  if (!out) return KS_EINVAL;
  *out = nullptr;
  if (!cfg || cfg->max_num_batched_tokens < 1 || cfg->max_num_seqs < 1 || cfg->block_size < 1 || cfg->num_blocks < 1 ||
      cfg->disk_blocks < 0 || (cfg->enable_prefix_cache != 0 && cfg->enable_prefix_cache != 1))
    return KS_EINVAL;
  ks_sched* s = new (std::nothrow) ks_sched();
  if (!s) return KS_ENOMEM;
  s->cfg = *cfg;
  s->free_blocks = cfg->num_blocks;
  *out = s;
  return KS_OK;
}

ks_status ks_sched_add_requests(ks_sched* s, int n, const double* arrival, const int32_t* prompt_len, const int32_t* max_new) {
  return ks_sched_add_prefixed_requests(s, n, arrival, prompt_len, max_new, nullptr, nullptr);
}

ks_status ks_sched_add_prefixed_requests(ks_sched* s, int n, const double* arrival, const int32_t* prompt_len,
                                         const int32_t* max_new, const int32_t* prefix_id, const int32_t* prefix_len) {
  if (!s || n < 0 || (n > 0 && (!arrival || !prompt_len || !max_new))) return KS_EINVAL;
  if ((prefix_id == nullptr) != (prefix_len == nullptr)) return KS_EINVAL;
  if (s->started) return KS_ESTATE;
  for (int i = 0; i < n; ++i) {
    if (!std::isfinite(arrival[i]) || prompt_len[i] < 1 || max_new[i] < 1) return KS_EINVAL;
    if (prefix_id && prefix_id[i] >= 0 && (prefix_len[i] < 0 || prefix_len[i] > prompt_len[i])) return KS_EINVAL;
    if (s->blocks_for((int64_t)prompt_len[i] + max_new[i]) > s->cfg.num_blocks) return KS_EINVAL;
  }
  if ((int64_t)s->arrival.size() + n > (int64_t)std::numeric_limits<int32_t>::max()) return KS_EINVAL;
  try {
    for (int i = 0; i < n; ++i) {
      s->arrival.push_back(arrival[i]);
      s->prompt.push_back(prompt_len[i]);
      s->max_new.push_back(max_new[i]);
      s->n_tok.push_back(prompt_len[i]);
      s->computed.push_back(0);
      s->generated.push_back(0);
      s->blocks.push_back(0);
      s->n_preempt.push_back(0);
      const bool pre = prefix_id && prefix_id[i] >= 0;
      s->prefix_id.push_back(pre ? prefix_id[i] : -1);
      s->prefix_len.push_back(pre ? prefix_len[i] : 0);
      s->registered.push_back(0);
      s->cached_tokens.push_back(0);
      s->held.emplace_back();
      s->first_token.push_back(std::numeric_limits<double>::quiet_NaN());
      s->finish.push_back(std::numeric_limits<double>::quiet_NaN());
    }
  } catch (const std::bad_alloc&) {
    return KS_ENOMEM;
  }
  return KS_OK;
}

ks_status ks_sched_step(ks_sched* s, double now, int32_t cap, int32_t* n_sched, int32_t* req, int32_t* n_new,
                        int32_t* hist, double* next_arrival) {
  if (!s || !n_sched || cap < 0 || std::isnan(now)) return KS_EINVAL;
  if (s->pending) return KS_ESTATE;
  if ((int64_t)cap < std::min<int64_t>(s->cfg.max_num_seqs, (int64_t)s->arrival.size()))
    return KS_EINVAL;                  // the caller's arrays might not hold the batch
  sched_form_batch(s, now);
  const int32_t n = (int32_t)s->b_req.size();
  *n_sched = n;
  for (int32_t k = 0; k < n; ++k) {
    if (req) req[k] = s->b_req[k];
    if (n_new) n_new[k] = s->b_new[k];
    if (hist) hist[k] = s->b_hist[k];
  }
  if (next_arrival) *next_arrival = sched_next_arrival(s);
  return KS_OK;
}

ks_status ks_sched_commit(ks_sched* s, double t_end) {
  if (!s || std::isnan(t_end)) return KS_EINVAL;
  if (!s->pending) return KS_ESTATE;
  sched_commit(s, t_end);
  return KS_OK;
}

ks_status ks_sched_results(ks_sched* s, double* first_token, double* finish, int32_t* n_preempt, int32_t* cached_tokens) {
  if (!s) return KS_EINVAL;
  const size_t n = s->arrival.size();
  if (first_token && n) memcpy(first_token, s->first_token.data(), n * sizeof(double));
  if (finish && n) memcpy(finish, s->finish.data(), n * sizeof(double));
  if (n_preempt && n) memcpy(n_preempt, s->n_preempt.data(), n * sizeof(int32_t));
  if (cached_tokens && n) memcpy(cached_tokens, s->cached_tokens.data(), n * sizeof(int32_t));
  return KS_OK;
}

ks_status ks_sched_get_stats(ks_sched* s, ks_sched_stats* out) {
  if (!s || !out) return KS_EINVAL;
  memset(out, 0, sizeof(*out));
  out->n_steps = s->n_steps;
  out->tokens_scheduled = s->tokens;
  out->n_preemptions = s->preemptions;
  out->n_requests = (int32_t)s->arrival.size();
  out->n_finished = s->n_finished;
  out->n_running = (int32_t)s->running.size();
  out->n_waiting = (int32_t)s->waiting.size();
  out->free_blocks = s->avail();
  out->gpu_hit_blocks = s->gpu_hits;
  out->disk_hit_blocks = s->disk_hits;
  out->evictions = s->evictions;
  return KS_OK;
}

ks_status ks_sched_destroy(ks_sched* s) {
  delete s;
  return KS_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// The closed loop.
namespace {

// One iteration's rows, packed for a single H2D copy.  Every array starts on a 16-byte boundary (the
// alignment KS_MEM_DEVICE asks for).  Buckets: GEMM, attention (all requests, or the prefill chunks when the model
// asks for the paper's fine model families), elementwise[, all-reduce][, LM head, decode attention].
constexpr int kSimBuckets = 6;
struct SimBucket {
  int family = 0, slot = KS_SLOT_FAMILY, n_cols = 0, cap_rows = 0;
  bool packed = false;                   // attention: columns packed every iteration at their actual length
  size_t col[3] = {}, mult = 0, off = 0;
};
struct Arena {
  char* host = nullptr;
  char* dev = nullptr;
  size_t bytes = 0;
  SimBucket bk[kSimBuckets];
  size_t out = 0;
  int n_bk = 3;
};

size_t a16(size_t x) { return (x + 15) & ~(size_t)15; }

}  // namespace

extern "C" ks_status ks_sim_run(ks_ctx* ctx, ks_sched* const* scheds, double* clock, int n_replicas,
                                const ks_model_desc* model, const ks_hw_spec* spec, ks_tier tier,
                                const ks_step_params* params, int64_t max_iters, int32_t* step_replica,
                                float* step_time, int64_t log_cap, int64_t* n_logged, ks_sim_stats* stats) {
  if (n_logged) *n_logged = 0;
  if (stats) memset(stats, 0, sizeof(*stats));
  if (!ctx || !scheds || !clock || n_replicas < 0 || !model || !spec || !params || log_cap < 0) return KS_EINVAL;
  if (log_cap > 0 && (!step_replica || !step_time)) return KS_EINVAL;
  const ks_model_desc& m = *model;
  if (m.n_layers < 1 || m.hidden < 1 || m.ffn < 1 || m.vocab < 1 || m.hq < 1 || m.hkv < 1 || m.head_dim < 1 || m.tp < 1 ||
      (m.dtype_bytes != 1 && m.dtype_bytes != 2 && m.dtype_bytes != 4) || (m.fine_slots != 0 && m.fine_slots != 1))
    return KS_EINVAL;
  for (int r = 0; r < n_replicas; ++r) {
    if (!scheds[r] || std::isnan(clock[r])) return KS_EINVAL;
    if (scheds[r]->pending) return KS_ESTATE;
    // int32 row columns: the largest value is tokens x max(2 ffn, hidden x dtype_bytes, ...)
    const int64_t T = scheds[r]->cfg.max_num_batched_tokens;
    const int64_t widest = std::max<int64_t>({(int64_t)m.ffn, (int64_t)m.hidden * m.dtype_bytes,
                                              (int64_t)(m.hq + m.hkv) * m.head_dim, (int64_t)2 * m.hkv * m.head_dim});
    if (T * widest > (int64_t)std::numeric_limits<int32_t>::max()) return KS_EUNSUPPORTED;
  }
  if (n_replicas == 0) return KS_OK;

  // PAPER.md:199 learns eta per kernel family — "GEMM, the LM head, attention prefill and decode, and the
  // elementwise and memory kernels": with fine_slots the LM-head row and the decode requests get buckets (and model
  // slots) of their own; the elementwise sub-operations keep one bucket (KS_MAX_BATCHES buckets per call).
  const bool fine = m.fine_slots != 0;
  Arena A;
  int64_t attn_rows = 0;
  for (int r = 0; r < n_replicas; ++r) attn_rows += scheds[r]->cfg.max_num_seqs;
  if (attn_rows > std::numeric_limits<int32_t>::max() / 8) return KS_EUNSUPPORTED;
  enum { B_GEMM = 0, B_ATTN = 1, B_ELEM = 2 };
  int B_AR = -1, B_LM = -1, B_DEC = -1, nb = 3;
  auto setb = [&A](int i, int family, int slot, int n_cols, int cap, bool packed) {
    A.bk[i].family = family; A.bk[i].slot = slot; A.bk[i].n_cols = n_cols; A.bk[i].cap_rows = cap; A.bk[i].packed = packed;
  };
  setb(B_GEMM, KS_FAM_GEMM, KS_SLOT_FAMILY, 3, (fine ? 4 : 5) * n_replicas, false);
  setb(B_ATTN, KS_FAM_ATTN, fine ? KS_SLOT_ATTN_PREFILL : KS_SLOT_FAMILY, 3, (int)attn_rows, true);
  setb(B_ELEM, KS_FAM_ELEMWISE, KS_SLOT_FAMILY, 2, 6 * n_replicas, false);
  if (m.tp > 1) { B_AR = nb++; setb(B_AR, KS_FAM_ALLREDUCE, KS_SLOT_FAMILY, 2, n_replicas, false); }
  if (fine) {
    B_LM = nb++; setb(B_LM, KS_FAM_GEMM, KS_SLOT_LM_HEAD, 3, n_replicas, false);
    B_DEC = nb++; setb(B_DEC, KS_FAM_ATTN, KS_SLOT_ATTN_DECODE, 3, (int)attn_rows, true);
  }
  A.n_bk = nb;
  // Fixed-size arrays first (a few rows per replica), the step times, and last the attention columns, which
  // are packed behind each other every iteration at their actual length: what an iteration reads is one
  // prefix of the arena, a few hundred KB at most.
  size_t at = 0;
  size_t packed_cap = 0;
  for (int f = 0; f < nb; ++f) {
    SimBucket& k = A.bk[f];
    if (!k.packed) {
      for (int c = 0; c < k.n_cols; ++c) { k.col[c] = at; at = a16(at + (size_t)k.cap_rows * 4); }
      k.mult = at; at = a16(at + (size_t)k.cap_rows * 4);
    } else {
      packed_cap += 4 * a16((size_t)k.cap_rows * 4);
    }
    k.off = at; at = a16(at + (size_t)(n_replicas + 1) * 4);
  }
  A.out = at; at = a16(at + (size_t)n_replicas * 4);
  const size_t attn_base = at;
  at += packed_cap;
  A.bytes = at;

  cudaStream_t st = ks_internal_stream(ctx);
  if (ks_internal_set_device(ctx) != cudaSuccess) return KS_ECUDA;
  if (cudaMallocHost((void**)&A.host, A.bytes) != cudaSuccess) { cudaGetLastError(); return KS_ENOMEM; }
  if (cudaMalloc((void**)&A.dev, A.bytes) != cudaSuccess) { cudaGetLastError(); cudaFreeHost(A.host); return KS_ENOMEM; }
  memset(A.host, 0, A.bytes);

  // Pinned host memory is addressable from the device (unified addressing), and an iteration is bound by
  // launch and copy latency, not bandwidth: the step times are always written straight into the pinned arena,
  // and an iteration whose rows fit 256 KB is also read in place (measured 47 vs 55 us per iteration); a
  // larger one is moved by one DMA copy of exactly the bytes in use.
  char* out_base = A.host;
  std::vector<int> active;
  active.reserve(n_replicas);
  ks_status rc = KS_OK;
  int64_t iters = 0, logged = 0, steps = 0, rows_total = 0, inst_total = 0;
  const int L = m.n_layers;
  // Per-GPU shapes under tensor parallelism (the all-reduces "combine partial activations
  // across the P shards"; Q20): attention heads and FFN columns are split P ways (ceil; KV heads
  // are replicated once P exceeds their number), QKV / Gate-Up are column-parallel (N / P), O / Down
  // row-parallel (K / P), the LM head vocabulary-parallel; norms and the embedding see the full hidden size.
  const int32_t P = m.tp;
  const int32_t hq_p = (m.hq + P - 1) / P, hkv_p = (m.hkv + P - 1) / P;
  const int32_t ffn_p = (m.ffn + P - 1) / P, vocab_p = (m.vocab + P - 1) / P;
  const int32_t qkv_n = (hq_p + 2 * hkv_p) * m.head_dim;
  auto I = [&A](size_t off) { return reinterpret_cast<int32_t*>(A.host + off); };

  double t_host = 0, t_enq = 0, t_wait = 0, t_commit = 0;
  auto tnow = [] { return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count(); };
  while (max_iters <= 0 || iters < max_iters) {
    const double tt0 = tnow();
    active.clear();
    int n_rows[kSimBuckets] = {0, 0, 0, 0, 0, 0};
    for (int f = 0; f < nb; ++f) I(A.bk[f].off)[0] = 0;
    // pass 1: every unfinished replica forms its batch
    int64_t attn_total[2] = {0, 0};                  // requests that go to bucket B_ATTN / B_DEC
    for (int r = 0; r < n_replicas; ++r) {
      ks_sched* s = scheds[r];
      if (sched_done(s)) continue;
      sched_form_batch(s, clock[r]);
      while (s->b_req.empty()) {                    // idle: the clock jumps to the next arrival
        const double nxt = sched_next_arrival(s);
        if (!std::isfinite(nxt)) break;
        clock[r] = std::max(clock[r], nxt);
        sched_form_batch(s, clock[r]);
      }
      if (s->b_req.empty()) continue;
      active.push_back(r);
      for (int32_t v : s->b_new) attn_total[(fine && v == 1) ? 1 : 0] += 1;
    }
    const int n_act = (int)active.size();
    if (n_act == 0) break;
    // pass 2: the batches' rows; the attention columns are packed at their actual length
    size_t pk = attn_base;
    for (int f = 0; f < nb; ++f) {
      SimBucket& k = A.bk[f];
      if (!k.packed) continue;
      const size_t stride = a16((size_t)attn_total[f == B_DEC ? 1 : 0] * 4);
      for (int c = 0; c < 3; ++c) k.col[c] = pk + (size_t)c * stride;
      k.mult = pk + 3 * stride;
      pk += 4 * stride;
    }
    const size_t in_bytes = pk;
    const bool in_place = in_bytes <= (256u << 10);
    char* in_base = in_place ? A.host : A.dev;
    for (int ai = 0; ai < n_act; ++ai) {
      ks_sched* s = scheds[active[ai]];
      // rows of this step: dense kernels at the total token count, attention per request
      int32_t T = 0;
      for (int32_t v : s->b_new) T += v;
      const int32_t n_seq = (int32_t)s->b_req.size();
      {
        const int32_t gM[5] = {T, T, T, T, n_seq};
        const int32_t gN[5] = {qkv_n, m.hidden, 2 * ffn_p, m.hidden, vocab_p};
        const int32_t gK[5] = {m.hidden, hq_p * m.head_dim, m.hidden, ffn_p, m.hidden};
        for (int j = 0; j < 5; ++j) {
          const int f = (fine && j == 4) ? B_LM : B_GEMM;     // the LM head: a GEMM-shaped row with its own model
          const int k = n_rows[f]++;
          I(A.bk[f].col[0])[k] = gM[j]; I(A.bk[f].col[1])[k] = gN[j]; I(A.bk[f].col[2])[k] = gK[j];
          I(A.bk[f].mult)[k] = j < 4 ? L : 1;
        }
      }
      for (int32_t j = 0; j < n_seq; ++j) {
        const int f = (fine && s->b_new[j] == 1) ? B_DEC : B_ATTN;   // decode: one new token over the cached context
        const int k = n_rows[f]++;
        I(A.bk[f].col[0])[k] = 1; I(A.bk[f].col[1])[k] = s->b_new[j]; I(A.bk[f].col[2])[k] = s->b_hist[j] + s->b_new[j];
        I(A.bk[f].mult)[k] = L;
      }
      {
        int k = n_rows[B_ELEM];
        const int32_t width[6] = {m.hidden, m.hidden, (hq_p + hkv_p) * m.head_dim, 2 * hkv_p * m.head_dim, ffn_p, m.hidden};
        const int32_t sub[6] = {4, 0, 2, 3, 1, 0};   // embedding, RMSNorm, RoPE, KV write, SiLU*Mul, final RMSNorm
        const int32_t mu[6] = {1, L, L, L, L, 1};
        for (int j = 0; j < 6; ++j, ++k) {
          I(A.bk[B_ELEM].col[0])[k] = T * width[j]; I(A.bk[B_ELEM].col[1])[k] = sub[j]; I(A.bk[B_ELEM].mult)[k] = mu[j];
        }
        n_rows[B_ELEM] = k;
      }
      if (B_AR >= 0) {
        const int k = n_rows[B_AR]++;
        I(A.bk[B_AR].col[0])[k] = T * m.hidden * m.dtype_bytes; I(A.bk[B_AR].col[1])[k] = m.tp; I(A.bk[B_AR].mult)[k] = 2 * L;
      }
      for (int f = 0; f < nb; ++f) I(A.bk[f].off)[ai + 1] = n_rows[f];
      inst_total += (int64_t)L * (4 + n_seq + 4 + (B_AR >= 0 ? 2 : 0)) + 3;
    }

    const double tt1 = tnow();
    // one copy in, one pass of the hot path on device pointers, one copy out
    if (!in_place && cudaMemcpyAsync(A.dev, A.host, in_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) { rc = KS_ECUDA; break; }
    ks_desc_batch b[kSimBuckets];
    const int32_t* offs[kSimBuckets];
    memset(b, 0, sizeof(b));
    for (int f = 0; f < nb; ++f) {
      const SimBucket& k = A.bk[f];
      b[f].family = k.family;
      b[f].model_slot = k.slot;
      b[f].n = n_rows[f];
      b[f].col_dtype = KS_COL_I32;
      b[f].dtype_bytes = m.dtype_bytes;
      b[f].n_cols = k.n_cols;
      if (k.family == KS_FAM_ATTN) { b[f].attn_hq = hq_p; b[f].attn_hkv = hkv_p; b[f].attn_head_dim = m.head_dim; }
      for (int c = 0; c < k.n_cols; ++c) b[f].cols[c] = in_base + k.col[c];
      b[f].mult = reinterpret_cast<const int32_t*>(in_base + k.mult);
      offs[f] = reinterpret_cast<const int32_t*>(in_base + k.off);
      rows_total += n_rows[f];
    }
    rc = ks_run_steps(ctx, b, offs, nb, spec, 1, tier, n_act, params, nullptr, 0, KS_MEM_DEVICE, nullptr,
                      reinterpret_cast<float*>(out_base + A.out), nullptr);
    if (rc != KS_OK) break;
    const double tt2 = tnow();
    if (cudaStreamSynchronize(st) != cudaSuccess) { rc = KS_ECUDA; break; }

    const double tt3 = tnow();
    const float* t_step = reinterpret_cast<const float*>(A.host + A.out);
    for (int a = 0; a < n_act; ++a) {
      const int r = active[a];
      clock[r] += (double)t_step[a];                 // completion at now + t_step
      sched_commit(scheds[r], clock[r]);
      if (logged < log_cap) { step_replica[logged] = r; step_time[logged] = t_step[a]; ++logged; }
    }
    steps += n_act;
    ++iters;
    const double tt4 = tnow();
    t_host += tt1 - tt0; t_enq += tt2 - tt1; t_wait += tt3 - tt2; t_commit += tt4 - tt3;
  }

  if (rc != KS_OK) {
    cudaStreamSynchronize(st);
    cudaGetLastError();
  }
  cudaFree(A.dev);
  cudaFreeHost(A.host);
  if (n_logged) *n_logged = logged;
  if (stats) {
    stats->iterations = iters; stats->steps = steps; stats->rows = rows_total; stats->kernel_instances = inst_total;
    stats->schedule_s = t_host; stats->enqueue_s = t_enq; stats->wait_s = t_wait; stats->commit_s = t_commit;
  }
  return rc;
}
