// ks_api.cu — the C ABI of libks (include/ks.h): context, head/grid loading (host-side operand
// image construction), argument validation, host<->device staging, kernel dispatch.
// No arithmetic of the method runs on the host; there is no CPU fallback.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>
#include <vector>

#include "ks_internal.h"

namespace {

struct HeadState {
  bool loaded = false;
  bool bounded = false;      // the family's Tier-A head is the bounded analytical form (host-resident weights)
  KsBoundedDev bw;
  int n_in = 0, h = 0;
  void* w1_img = nullptr;
  void* w2_img = nullptr;
  float* w3 = nullptr;
  float* b2 = nullptr;
  float b3 = 0.0f;
  int members = 1;           // > 1: MLP ensemble packed as one head of width h (Q17)
  float b3m[KS_MAX_ENSEMBLE] = {};
  int out_mode = KS_HEAD_UTILISATION;   // what z means (ks_set_head_output)
};

struct GridState {
  bool loaded = false;
  KsGridDev dev;
  KsTierBGrid tb;            // the same grid in the form the GEMM/attention Tier-B kernel takes (ks_tierb.cu)
  float* values = nullptr;
};

}  // namespace

struct ks_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  int num_sms = 0;
  bool sticky = false;
  int gelu_mode = 0;
  int64_t launches = 0;
  HeadState heads[KS_MAX_MODEL_SLOTS];   // by model slot (include/ks.h: ks_model_slot), not by decode family
  GridState grids[KS_MAX_MODEL_SLOTS];
  // grow-only device workspace with a bump pointer (host-space staging, internal latencies)
  char* ws = nullptr;
  size_t ws_cap = 0, ws_used = 0;
  // host-space pipeline of ks_run_steps: bucket b's H2D copies run on `h2d` while bucket b-1 is
  // predicted on `stream` and bucket b-2's latencies return on `d2h` (created on first use)
  cudaStream_t h2d = nullptr, d2h = nullptr;
  cudaEvent_t ev_in[KS_MAX_BATCHES] = {}, ev_out[KS_MAX_BATCHES] = {}, ev_start = nullptr;
};

cudaStream_t ks_internal_stream(ks_ctx* c) { return c->stream; }
cudaError_t ks_internal_set_device(ks_ctx* c) { return cudaSetDevice(c->device); }

namespace {

const int kFamCols[KS_FAM_COUNT] = {3, 10, 3, 2, 2};

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// the model slot that prices a bucket: its own, or the one numbered like its family
inline int slot_of(const ks_desc_batch& k) { return k.model_slot == KS_SLOT_FAMILY ? k.family : k.model_slot; }
inline bool slot_ok(int slot) { return slot >= 0 && slot < KS_MAX_MODEL_SLOTS; }

ks_status cuda_fail(ks_ctx* c) {
  if (c) c->sticky = true;
  return KS_ECUDA;
}

#define KS_CUDA(ctx, call)                       \
  do {                                           \
    if ((call) != cudaSuccess) return cuda_fail(ctx); \
  } while (0)

ks_status ws_reserve(ks_ctx* c, size_t bytes) {
  c->ws_used = 0;
  if (bytes <= c->ws_cap) return KS_OK;
  if (c->ws) {
    KS_CUDA(c, cudaStreamSynchronize(c->stream));
    KS_CUDA(c, cudaFree(c->ws));
    c->ws = nullptr;
    c->ws_cap = 0;
  }
  const size_t cap = align_up(bytes + bytes / 8, 1 << 20);
  if (cudaMalloc(reinterpret_cast<void**>(&c->ws), cap) != cudaSuccess) {
    cudaGetLastError();
    c->ws = nullptr;
    return KS_ENOMEM;
  }
  c->ws_cap = cap;
  return KS_OK;
}

void* ws_take(ks_ctx* c, size_t bytes) {
  void* p = c->ws + c->ws_used;
  c->ws_used += align_up(bytes, 256);
  return p;
}

ks_status pipeline_init(ks_ctx* c) {
  if (c->h2d) return KS_OK;
  KS_CUDA(c, cudaStreamCreateWithFlags(&c->h2d, cudaStreamNonBlocking));
  KS_CUDA(c, cudaStreamCreateWithFlags(&c->d2h, cudaStreamNonBlocking));
  for (int b = 0; b < KS_MAX_BATCHES; ++b) {
    KS_CUDA(c, cudaEventCreateWithFlags(&c->ev_in[b], cudaEventDisableTiming));
    KS_CUDA(c, cudaEventCreateWithFlags(&c->ev_out[b], cudaEventDisableTiming));
  }
  KS_CUDA(c, cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming));
  return KS_OK;
}

// fp32 -> bf16 bits, round to nearest even (NaN kept quiet)
uint16_t f32_to_bf16_bits(float f) {
  uint32_t u;
  memcpy(&u, &f, 4);
  if ((u & 0x7f800000u) == 0x7f800000u && (u & 0x007fffffu)) return (uint16_t)((u >> 16) | 0x40u);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}
float bf16_bits_to_f32(uint16_t b) {
  uint32_t u = (uint32_t)b << 16;
  float f;
  memcpy(&f, &u, 4);
  return f;
}

KsFastDiv make_fastdiv(uint32_t d) {
  KsFastDiv f;
  if (d < 1) d = 1;
  f.d = d;
  f.pad = 0;
  uint32_t l = 0;
  while ((1ull << l) < d) ++l;                       // ceil(log2 d); d = 1 -> l = 0, mul = 2^31
  f.mul = (uint32_t)(((1ull << (31 + l)) + d - 1) / d);
  f.shr = l;
  return f;
}

bool spec_ok(const ks_hw_spec& s) {
  if (!(s.peak_flops > 0.0f) || !(s.peak_bw > 0.0f) || !isfinite(s.peak_flops) || !isfinite(s.peak_bw)) return false;
  if (s.n_sm < 1 || s.ctas_per_sm < 1 || s.tile_m < 1 || s.tile_n < 1 || s.ew_elems_per_cta < 1) return false;
  if ((long long)s.n_sm * s.ctas_per_sm > 0x7fffffffll) return false;
  if (!(s.l2_bytes >= 0.0f) || !(s.t0 >= 0.0f) || !isfinite(s.t0)) return false;
  if (!(s.ar_alpha0 >= 0.0f) || !isfinite(s.ar_alpha0) || !(s.ar_beta_eff > 0.0f) || !isfinite(s.ar_beta_eff)) return false;
  return true;
}

KsSpecDev make_spec_dev(const ks_hw_spec& s) {
  KsSpecDev d;
  const uint32_t slots = (uint32_t)s.n_sm * (uint32_t)s.ctas_per_sm;
  d.inv_peak_flops = (float)(1.0 / (double)s.peak_flops);
  d.inv_peak_bw = (float)(1.0 / (double)s.peak_bw);
  d.t0 = s.t0;
  d.inv_t0 = s.t0 > 0.0f ? (float)(1.0 / (double)s.t0) : INFINITY;
  d.l2_bytes = s.l2_bytes;
  d.lg_ridge = (float)log2((double)s.peak_flops / (double)s.peak_bw);
  d.inv_slots = (float)(1.0 / (double)slots);
  d.slots_f = (float)slots;
  d.tile_m = make_fastdiv((uint32_t)s.tile_m);
  d.tile_n = make_fastdiv((uint32_t)s.tile_n);
  d.ew = make_fastdiv((uint32_t)s.ew_elems_per_cta);
  d.slots = make_fastdiv(slots);
  d.ar_alpha0 = s.ar_alpha0;
  d.ar_inv_beta = (float)(1.0 / (double)s.ar_beta_eff);
  d.pad0 = d.pad1 = 0.0f;
  return d;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// validation shared by predict / run_steps.  `device_ptrs`: enforce 16-byte alignment.
ks_status validate_batches(const ks_ctx* c, const ks_desc_batch* batches, int n_batches, const ks_hw_spec* specs,
                           int n_specs, int tier, bool device_ptrs) {
  if (!c) return KS_EINVAL;
  if (n_batches < 0 || n_batches > KS_MAX_BATCHES || n_specs < 0) return KS_EINVAL;
  if (n_batches > 0 && !batches) return KS_EINVAL;
  if (n_specs > 0 && !specs) return KS_EINVAL;
  if (tier != KS_TIER_NONE && tier != KS_TIER_A && tier != KS_TIER_B && tier != KS_TIER_B_ROUTED) return KS_EINVAL;
  for (int s = 0; s < n_specs; ++s)
    if (!spec_ok(specs[s])) return KS_EINVAL;
  for (int b = 0; b < n_batches; ++b) {
    const ks_desc_batch& k = batches[b];
    if (k.family < 0 || k.family >= KS_FAM_COUNT || k.n < 0) return KS_EINVAL;
    if (k.col_dtype != KS_COL_I32 && k.col_dtype != KS_COL_F32) return KS_EINVAL;
    if (k.dtype_bytes != 1 && k.dtype_bytes != 2 && k.dtype_bytes != 4) return KS_EINVAL;
    if (k.n_cols != kFamCols[k.family]) return KS_EINVAL;
    if (k.family == KS_FAM_ATTN && (k.attn_hq < 1 || k.attn_hkv < 1 || k.attn_head_dim < 1)) return KS_EINVAL;
    if (k.n > 0)
      for (int col = 0; col < k.n_cols; ++col) {
        if (!k.cols[col]) return KS_EINVAL;
        if (device_ptrs && !aligned16(k.cols[col])) return KS_EINVAL;
      }
    if (k.model_slot != KS_SLOT_FAMILY && !slot_ok(k.model_slot)) return KS_EINVAL;
    if (k.family == KS_FAM_ALLREDUCE) continue;               // Eq. 3 needs neither head nor grid
    if ((tier == KS_TIER_A || tier == KS_TIER_B_ROUTED) && !c->heads[slot_of(k)].loaded) return KS_ESTATE;
    if ((tier == KS_TIER_B || tier == KS_TIER_B_ROUTED) && !c->grids[slot_of(k)].loaded) return KS_ESTATE;
  }
  return KS_OK;
}

struct DevOut {
  float* lat = nullptr;
  int32_t* tiles = nullptr;
  int32_t* waves = nullptr;
  float* troof = nullptr;
};

KsBucketDev make_bucket_dev(const ks_desc_batch& k, const void* const* cols, const DevOut& o, long long spec0) {
  KsBucketDev d;
  memset(&d, 0, sizeof(d));
  for (int c = 0; c < k.n_cols; ++c) d.cols[c] = cols[c];
  const long long off = spec0 * (long long)k.n;
  d.lat = o.lat ? o.lat + off : nullptr;
  d.tiles = o.tiles ? o.tiles + off : nullptr;
  d.waves = o.waves ? o.waves + off : nullptr;
  d.troof = o.troof ? o.troof + off : nullptr;
  d.family = k.family;
  d.n = k.n;
  d.col_f32 = k.col_dtype == KS_COL_F32 ? 1 : 0;
  d.s = k.dtype_bytes;
  d.hq = k.attn_hq;
  d.hkv = k.attn_hkv;
  d.hd = k.attn_head_dim;
  d.n_cols = k.n_cols;
  return d;
}

// Density routing scratch: per bucket a row list (n ints) and its length (one int, in its own 256-byte slot).
struct RouteBuf {
  int32_t* idx = nullptr;
  int32_t* count = nullptr;
};
size_t route_need(const ks_desc_batch* batches, int n_batches, int tier) {
  size_t need = 0;
  if (tier != KS_TIER_B_ROUTED) return 0;
  for (int b = 0; b < n_batches; ++b)
    if (batches[b].family != KS_FAM_ALLREDUCE) need += align_up((size_t)batches[b].n * 4, 256) + 256;
  return need;
}
void route_take(ks_ctx* c, const ks_desc_batch* batches, int n_batches, int tier, RouteBuf* rb) {
  for (int b = 0; b < n_batches; ++b) {
    rb[b] = RouteBuf();
    if (tier != KS_TIER_B_ROUTED || batches[b].family == KS_FAM_ALLREDUCE) continue;
    rb[b].idx = static_cast<int32_t*>(ws_take(c, (size_t)batches[b].n * 4));
    rb[b].count = static_cast<int32_t*>(ws_take(c, 4));
  }
}

// Enqueue S1-S5 for device-resident columns/outputs.  Arguments are already validated.
// tier == KS_TIER_B_ROUTED: pass 1 = the Tier-B kernel on every row, which also lists
// the rows outside the measured hull in rb[b]; pass 2 = the family's Tier-A head (tcgen05 MLP kernel
// or bounded form) on that row list, overwriting those rows' latencies.
ks_status predict_device(ks_ctx* c, const ks_desc_batch* batches, const void* const (*cols)[KS_MAX_COLS], int n_batches,
                         const ks_hw_spec* specs, int n_specs, int tier_in, const DevOut* outs,
                         const RouteBuf* rb = nullptr) {
  const bool routed = tier_in == KS_TIER_B_ROUTED;
  if (routed && !rb) return KS_EINVAL;
  for (int pass = 0; pass < (routed ? 2 : 1); ++pass) {
  const int tier = routed ? (pass == 0 ? KS_TIER_B : KS_TIER_A) : tier_in;
  const bool lists = routed && pass == 1;
  for (int s0 = 0; s0 < n_specs; s0 += KS_MAX_SPECS_PER_LAUNCH) {
    const int ns = n_specs - s0 < KS_MAX_SPECS_PER_LAUNCH ? n_specs - s0 : KS_MAX_SPECS_PER_LAUNCH;
    // a small Tier-NONE call with several buckets: one launch for all of them
    if (tier == KS_TIER_NONE && !lists && !routed && n_batches > 1) {
      long long total = 0;
      int nonempty = 0;
      for (int b = 0; b < n_batches; ++b) { total += batches[b].n; nonempty += batches[b].n > 0; }
      if (nonempty > 1 && total <= KS_STREAM_SMALL_MAX_ROWS) {
        KsStreamSmallParams p;
        memset(&p, 0, sizeof(p));
        for (int b = 0; b < n_batches; ++b) {
          p.bk[b] = make_bucket_dev(batches[b], cols[b], outs[b], s0);
          p.row_begin[b + 1] = p.row_begin[b] + batches[b].n;
        }
        p.n_buckets = n_batches;
        p.n_specs = ns;
        for (int s = 0; s < ns; ++s) p.specs.s[s] = make_spec_dev(specs[s0 + s]);
        KS_CUDA(c, ks_launch_stream_small(p, c->stream));
        c->launches += 1;
        continue;
      }
    }
    // Tier B, GEMM and attention buckets: ONE persistent launch for all of them (per column type)
    bool tb_done[KS_MAX_BATCHES] = {false};
    if (tier == KS_TIER_B) {
      for (int f32 = 0; f32 < 2; ++f32) {
        int b0 = 0;
        while (b0 < n_batches) {
          KsTierBParams p;
          memset(&p, 0, sizeof(p));
          int nb = 0;
          for (; b0 < n_batches && nb < KS_TIERB_MAX_BUCKETS; ++b0) {
            const ks_desc_batch& k = batches[b0];
            if ((k.family != KS_FAM_GEMM && k.family != KS_FAM_ATTN) || (k.col_dtype == KS_COL_F32) != (f32 == 1)) continue;
            tb_done[b0] = true;
            if (k.n == 0) continue;
            p.bk[nb] = make_bucket_dev(k, cols[b0], outs[b0], s0);
            p.grid[nb] = c->grids[slot_of(k)].tb;
            if (routed && s0 == 0) {                      // the hull test depends on the row only: list it once
              KS_CUDA(c, cudaMemsetAsync(rb[b0].count, 0, 4, c->stream));
              p.grid[nb].route_idx = rb[b0].idx;
              p.grid[nb].route_count = rb[b0].count;
            }
            ++nb;
          }
          if (nb == 0) continue;
          p.n_buckets = nb;
          p.n_specs = ns;
          for (int s = 0; s < ns; ++s) p.specs.s[s] = make_spec_dev(specs[s0 + s]);
          KS_CUDA(c, ks_launch_tierb(p, c->num_sms, c->stream));
          c->launches += 1;
        }
      }
    }
    for (int b = 0; b < n_batches; ++b) {               // streaming kernels: Tier NONE / B, and Eq. 3 rows under any tier
      if (tb_done[b]) continue;
      const bool ar = batches[b].family == KS_FAM_ALLREDUCE;
      if (ar && lists) continue;                        // Eq. 3 rows were finished by pass 1
      const bool bnd = tier == KS_TIER_A && !ar && c->heads[slot_of(batches[b])].bounded;
      if (batches[b].n == 0 || (tier == KS_TIER_A && !ar && !bnd)) continue;
      {
        KsStreamParams p;
        memset(&p, 0, sizeof(p));
        p.bk = make_bucket_dev(batches[b], cols[b], outs[b], s0);
        if (lists) { p.bk.idx = rb[b].idx; p.bk.count = rb[b].count; }
        if (tier == KS_TIER_B && !ar) p.grid = c->grids[slot_of(batches[b])].dev;
        if (routed && pass == 0 && !ar && s0 == 0) {    // the hull test depends on the row only: list it once
          KS_CUDA(c, cudaMemsetAsync(rb[b].count, 0, 4, c->stream));
          p.grid.route_idx = rb[b].idx;
          p.grid.route_count = rb[b].count;
        }
        p.n_specs = ns;
        p.tier = ar ? KS_TIER_NONE : bnd ? KS_TIER_BOUNDED : tier;
        if (bnd) p.bounded = c->heads[slot_of(batches[b])].bw;
        p.spec_stride = batches[b].n;
        for (int s = 0; s < ns; ++s) p.specs.s[s] = make_spec_dev(specs[s0 + s]);
        KS_CUDA(c, ks_launch_stream(p, c->num_sms, c->stream));
        c->launches += 1;
      }
    }
    if (tier == KS_TIER_A) {
      // group buckets by head dimensions; one persistent launch per group of <= 4 buckets
      bool done[KS_MAX_BATCHES] = {false};
      for (int b = 0; b < n_batches; ++b) {
        if (batches[b].family == KS_FAM_ALLREDUCE || c->heads[slot_of(batches[b])].bounded) done[b] = true;
        if (done[b] || batches[b].n == 0) { done[b] = true; continue; }
        const HeadState& h0 = c->heads[slot_of(batches[b])];
        KsMlpParams p;
        memset(&p, 0, sizeof(p));
        int nb = 0, tiles = 0;
        for (int q = b; q < n_batches && nb < KS_MLP_MAX_BUCKETS; ++q) {
          if (done[q] || batches[q].n == 0 || batches[q].family == KS_FAM_ALLREDUCE ||
              c->heads[slot_of(batches[q])].bounded) continue;
          const HeadState& hq = c->heads[slot_of(batches[q])];
          if (hq.n_in != h0.n_in || hq.h != h0.h) continue;
          p.bk[nb] = make_bucket_dev(batches[q], cols[q], outs[q], s0);
          if (lists) { p.bk[nb].idx = rb[q].idx; p.bk[nb].count = rb[q].count; }
          p.head[nb].w1_img = hq.w1_img;
          p.head[nb].w2_img = hq.w2_img;
          p.head[nb].w3 = hq.w3;
          p.head[nb].b2 = hq.b2;
          p.head[nb].b3 = hq.b3;
          p.head[nb].members = hq.members;
          // eta = out_add + exp(max(out_sgn * z, out_lo)): 1 + exp(-z) (utilisation) or exp(max(z, 0)) (log eta)
          const bool log_eta = hq.out_mode == KS_HEAD_LOG_ETA;
          p.head[nb].out_sgn = log_eta ? 1.0f : -1.0f;
          p.head[nb].out_lo = log_eta ? 0.0f : -INFINITY;
          p.head[nb].out_add = log_eta ? 0.0f : 1.0f;
          if (hq.members > 1) p.any_ens = 1;
          for (int m = 0; m < KS_MAX_ENSEMBLE; ++m) p.head[nb].b3m[m] = hq.b3m[m];
          p.tile_begin[nb] = tiles;
          tiles += (batches[q].n + 127) / 128;
          done[q] = true;
          ++nb;
        }
        p.tile_begin[nb] = tiles;
        p.n_buckets = nb;
        p.n_specs = ns;
        p.gelu_mode = c->gelu_mode;
        for (int s = 0; s < ns; ++s) p.specs.s[s] = make_spec_dev(specs[s0 + s]);
        KS_CUDA(c, ks_launch_mlp(p, h0.n_in, h0.h, c->num_sms, c->stream));
        c->launches += 1;
      }
    }
  }
  }
  return KS_OK;
}

}  // namespace

// =================================================================== extern "C" entry points
extern "C" {

const char* ks_status_string(ks_status s) {
  switch (s) {
    case KS_OK: return "KS_OK";
    case KS_EINVAL: return "KS_EINVAL";
    case KS_ENOMEM: return "KS_ENOMEM";
    case KS_ECUDA: return "KS_ECUDA";
    case KS_ESTATE: return "KS_ESTATE";
    case KS_EUNSUPPORTED: return "KS_EUNSUPPORTED";
    case KS_ELIMIT: return "KS_ELIMIT";
  }
  return "KS_?";
}

ks_status ks_create(ks_ctx** out, int device, void* cuda_stream) {
  if (!out) return KS_EINVAL;
  *out = nullptr;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) { cudaGetLastError(); return KS_ECUDA; }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaGetLastError(); return KS_ECUDA; }
  if (prop.major != 10) return KS_ECUDA;            // kernels are built for sm_100a only; no fallback
  if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return KS_ECUDA; }
  ks_ctx* c = new (std::nothrow) ks_ctx();
  if (!c) return KS_ENOMEM;
  c->device = device;
  c->stream = static_cast<cudaStream_t>(cuda_stream);
  c->num_sms = prop.multiProcessorCount;
  *out = c;
  return KS_OK;
}

ks_status ks_destroy(ks_ctx* c) {
  if (!c) return KS_OK;
  cudaSetDevice(c->device);
  cudaStreamSynchronize(c->stream);
  for (int f = 0; f < KS_MAX_MODEL_SLOTS; ++f) {
    cudaFree(c->heads[f].w1_img);
    cudaFree(c->heads[f].w2_img);
    cudaFree(c->heads[f].w3);
    cudaFree(c->heads[f].b2);
    cudaFree(c->grids[f].values);
  }
  cudaFree(c->ws);
  if (c->h2d) cudaStreamDestroy(c->h2d);
  if (c->d2h) cudaStreamDestroy(c->d2h);
  for (int b = 0; b < KS_MAX_BATCHES; ++b) {
    if (c->ev_in[b]) cudaEventDestroy(c->ev_in[b]);
    if (c->ev_out[b]) cudaEventDestroy(c->ev_out[b]);
  }
  if (c->ev_start) cudaEventDestroy(c->ev_start);
  cudaGetLastError();
  delete c;
  return KS_OK;
}

ks_status ks_get_launch_count(ks_ctx* c, int64_t* out) {
  if (!c || !out) return KS_EINVAL;
  *out = c->launches;
  return KS_OK;
}

ks_status ks_set_head_output(ks_ctx* c, int slot, ks_head_output mode) {
  if (!c || !slot_ok(slot) || (mode != KS_HEAD_UTILISATION && mode != KS_HEAD_LOG_ETA)) return KS_EINVAL;
  HeadState& hs = c->heads[slot];
  if (!hs.loaded) return KS_ESTATE;
  if (hs.bounded || hs.members > 1) return KS_EUNSUPPORTED;
  hs.out_mode = mode;                                // read when a launch is built: no device state to update
  return KS_OK;
}

ks_status ks_set_gelu_mode(ks_ctx* c, int mode) {
  if (!c || (mode != 0 && mode != 1)) return KS_EINVAL;
  c->gelu_mode = mode;
  return KS_OK;
}

namespace {

// Builds the operand images of a dense head n_in -> H -> H and installs it for `family`.  members > 1:
// the arrays hold an ensemble packed by ks_load_head_ensemble and b3m its per-member output biases.
ks_status install_head(ks_ctx* c, int slot, int n_in, int H, const float* W1, const float* b1,
                       const float* W2, const float* b2, const float* w3, float b3, int members, const float* b3m) {
  const int K1 = ks_mlp_k1(n_in);
  const int n_real = n_in == 32 ? 22 : n_in;          // features 22..31 are identically zero (Q2)
  const int bias_row = n_real;
  // UMMA operand images, K-major no-swizzle: element (n, k) at ((k/8) * H + n) * 8 + k % 8
  // (rows H + 16 .. H + 23 of the layer-2 image: one more K chunk with b2 hi / lo at the chunk positions of layer 1's
  // constant-1 feature columns -- the H = 256 kernel adds b2 with one K = 16 MMA against the A1 operand, ks_mlp_ws256.cu)
  std::vector<uint16_t> i1((size_t)K1 * H, 0), i2((size_t)(H + 24) * H, 0);
  auto at = [H](int n, int k) { return ((size_t)(k / 8) * H + n) * 8 + (k % 8); };
  for (int j = 0; j < H; ++j) {
    for (int k = 0; k < n_real; ++k) i1[at(j, k)] = f32_to_bf16_bits(W1[(size_t)k * H + j]);
    const uint16_t hi1 = f32_to_bf16_bits(b1[j]);
    i1[at(j, bias_row)] = hi1;
    i1[at(j, bias_row + 1)] = f32_to_bf16_bits(b1[j] - bf16_bits_to_f32(hi1));
    // the kernels produce 2 GELU(.) as hidden activation; the factor 1/2 lives in the next layer's
    // weights (a power-of-two scaling of a bf16 value is exact)
    for (int k = 0; k < H; ++k) i2[at(j, k)] = f32_to_bf16_bits(0.5f * bf16_bits_to_f32(f32_to_bf16_bits(W2[(size_t)k * H + j])));
    const uint16_t hi2 = f32_to_bf16_bits(b2[j]);
    i2[at(j, H)] = hi2;
    i2[at(j, H + 1)] = f32_to_bf16_bits(b2[j] - bf16_bits_to_f32(hi2));
    i2[at(j, H + 16 + bias_row % 8)] = hi2;
    i2[at(j, H + 16 + bias_row % 8 + 1)] = i2[at(j, H + 1)];
  }
  // layer 3 runs in fp32 on the CUDA cores; its weights are still bf16-rounded like the others
  std::vector<float> w3r(H);
  for (int j = 0; j < H; ++j) w3r[j] = 0.5f * bf16_bits_to_f32(f32_to_bf16_bits(w3[j]));

  KS_CUDA(c, cudaSetDevice(c->device));
  KS_CUDA(c, cudaStreamSynchronize(c->stream));       // nothing in flight may still read the old head
  HeadState& hs = c->heads[slot];
  cudaFree(hs.w1_img); cudaFree(hs.w2_img); cudaFree(hs.w3); cudaFree(hs.b2);
  hs = HeadState();
  void *d1 = nullptr, *d2 = nullptr, *d3 = nullptr, *d4 = nullptr;
  if (cudaMalloc(&d1, i1.size() * 2) != cudaSuccess || cudaMalloc(&d2, i2.size() * 2) != cudaSuccess ||
      cudaMalloc(&d3, (size_t)H * 4) != cudaSuccess || cudaMalloc(&d4, (size_t)H * 4) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(d1); cudaFree(d2); cudaFree(d3); cudaFree(d4);
    return KS_ENOMEM;
  }
  if (cudaMemcpy(d4, b2, (size_t)H * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(d1, i1.data(), i1.size() * 2, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(d2, i2.data(), i2.size() * 2, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(d3, w3r.data(), (size_t)H * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
    cudaFree(d1); cudaFree(d2); cudaFree(d3); cudaFree(d4);
    return cuda_fail(c);
  }
  hs.loaded = true;
  hs.n_in = n_in;
  hs.h = H;
  hs.w1_img = d1;
  hs.w2_img = d2;
  hs.w3 = static_cast<float*>(d3);
  hs.b2 = static_cast<float*>(d4);
  hs.b3 = b3;
  hs.members = members;
  for (int m = 0; m < members && m < KS_MAX_ENSEMBLE && b3m; ++m) hs.b3m[m] = b3m[m];
  return KS_OK;
}

}  // namespace

ks_status ks_load_heads(ks_ctx* c, int slot, int n_in, int h1, int h2, const float* W1, const float* b1,
                        const float* W2, const float* b2, const float* w3, float b3) {
  if (!c || !slot_ok(slot) || !W1 || !b1 || !W2 || !b2 || !w3) return KS_EINVAL;
  if (n_in <= 0 || h1 <= 0 || h2 <= 0) return KS_EINVAL;
  if (c->sticky) return KS_ECUDA;
  if ((n_in != 8 && n_in != 12 && n_in != 32) || h1 != h2 || (h1 != 64 && h1 != 128 && h1 != 256)) return KS_EUNSUPPORTED;
  return install_head(c, slot, n_in, h1, W1, b1, W2, b2, w3, b3, 1, nullptr);
}

ks_status ks_load_head_ensemble(ks_ctx* c, int slot, int n_in, int h, int n_members, const float* W1,
                                const float* b1, const float* W2, const float* b2, const float* w3, const float* b3) {
  if (!c || !slot_ok(slot) || !W1 || !b1 || !W2 || !b2 || !w3 || !b3)
    return KS_EINVAL;
  if (n_in <= 0 || h <= 0 || n_members <= 0) return KS_EINVAL;
  if (c->sticky) return KS_ECUDA;
  const int H = h * n_members;
  if ((n_in != 8 && n_in != 12 && n_in != 32) || n_members > KS_MAX_ENSEMBLE || (h != 32 && h != 64 && h != 128) ||
      (H != 64 && H != 128 && H != 256))
    return KS_EUNSUPPORTED;
  if (n_members == 1) return install_head(c, slot, n_in, h, W1, b1, W2, b2, w3, b3[0], 1, nullptr);
  // Pack the members side by side into one head of width H = k h: layer 1 concatenated along its outputs,
  // layer 2 block-diagonal (the zero blocks contribute exact zeros to the fp32 accumulators), layer 3
  // concatenated; the kernels close one dot product + sigmoid per member and average (Q17).
  std::vector<float> pW1((size_t)n_in * H), pb1(H), pW2((size_t)H * H, 0.0f), pb2(H), pw3(H);
  for (int m = 0; m < n_members; ++m) {
    const float* mW1 = W1 + (size_t)m * n_in * h;
    const float* mW2 = W2 + (size_t)m * h * h;
    for (int i = 0; i < n_in; ++i)
      for (int j = 0; j < h; ++j) pW1[(size_t)i * H + m * h + j] = mW1[(size_t)i * h + j];
    for (int i = 0; i < h; ++i)
      for (int j = 0; j < h; ++j) pW2[(size_t)(m * h + i) * H + m * h + j] = mW2[(size_t)i * h + j];
    for (int j = 0; j < h; ++j) {
      pb1[m * h + j] = b1[(size_t)m * h + j];
      pb2[m * h + j] = b2[(size_t)m * h + j];
      pw3[m * h + j] = w3[(size_t)m * h + j];
    }
  }
  return install_head(c, slot, n_in, H, pW1.data(), pb1.data(), pW2.data(), pb2.data(), pw3.data(), 0.0f,
                      n_members, b3);
}

ks_status ks_load_bounded_head(ks_ctx* c, int slot, int n_in, const float* w_gamma, float b_gamma,
                               const float* w_alpha, float b_alpha) {
  if (!c || !slot_ok(slot) || !w_gamma || !w_alpha) return KS_EINVAL;
  if (n_in <= 0 || !isfinite(b_gamma) || !isfinite(b_alpha)) return KS_EINVAL;
  if (n_in != 8 && n_in != 12 && n_in != 32) return KS_EUNSUPPORTED;    // before the arrays are read: their length is n_in
  for (int i = 0; i < n_in; ++i)
    if (!isfinite(w_gamma[i]) || !isfinite(w_alpha[i])) return KS_EINVAL;
  if (c->sticky) return KS_ECUDA;
  KS_CUDA(c, cudaSetDevice(c->device));
  KS_CUDA(c, cudaStreamSynchronize(c->stream));       // nothing in flight may still read an MLP head being replaced
  HeadState& hs = c->heads[slot];
  cudaFree(hs.w1_img); cudaFree(hs.w2_img); cudaFree(hs.w3); cudaFree(hs.b2);
  hs = HeadState();
  memset(&hs.bw, 0, sizeof(hs.bw));
  const int n_real = n_in == 32 ? KS_BOUNDED_NF : n_in;   // features 22..31 are identically zero (Q2)
  for (int i = 0; i < n_real; ++i) { hs.bw.w_gamma[i] = w_gamma[i]; hs.bw.w_alpha[i] = w_alpha[i]; }
  hs.bw.b_gamma = b_gamma;
  hs.bw.b_alpha = b_alpha;
  hs.loaded = true;
  hs.bounded = true;
  hs.n_in = n_in;
  return KS_OK;
}

ks_status ks_load_grid(ks_ctx* c, int slot, const int32_t dims[3], const float lo_log2[3],
                       const float hi_log2[3], const float* values) {
  if (!c || !slot_ok(slot) || !dims || !lo_log2 || !hi_log2 || !values) return KS_EINVAL;
  long long nodes = 1;
  for (int a = 0; a < 3; ++a) {
    if (dims[a] < 1 || dims[a] > KS_MAX_GRID_NODES) return KS_EINVAL;
    if (dims[a] > 1 && !(hi_log2[a] > lo_log2[a])) return KS_EINVAL;
    // axis values are int32: their log2 lies in [0, 31]; the kernels' exponent arithmetic is exact for |lo| <= 64
    if (dims[a] > 1 && !(lo_log2[a] >= -64.0f && hi_log2[a] <= 64.0f)) return KS_EINVAL;
    nodes *= dims[a];
  }
  if (nodes > KS_MAX_GRID_NODES) return KS_EINVAL;
  for (long long i = 0; i < nodes; ++i)
    if (!isfinite(values[i])) return KS_EINVAL;
  if (c->sticky) return KS_ECUDA;
  KS_CUDA(c, cudaSetDevice(c->device));
  KS_CUDA(c, cudaStreamSynchronize(c->stream));
  GridState& g = c->grids[slot];
  cudaFree(g.values);
  g = GridState();
  // bulk copies move multiples of 16 bytes.  Behind the last node: one plane + one row + two floats of zeros (the
  // Tier-B kernel reads the corners one node past an axis' end with weight exactly 0; they must be finite)
  const size_t tail = (size_t)(dims[0] > 1 ? dims[1] * dims[2] : 0) + (size_t)(dims[1] > 1 ? dims[2] : 0) + 2;
  const size_t padded = ((size_t)nodes + tail + 3) & ~(size_t)3;
  float* d = nullptr;
  if (cudaMalloc(reinterpret_cast<void**>(&d), padded * 4) != cudaSuccess) { cudaGetLastError(); return KS_ENOMEM; }
  KS_CUDA(c, cudaMemset(d, 0, padded * 4));
  KS_CUDA(c, cudaMemcpy(d, values, (size_t)nodes * 4, cudaMemcpyHostToDevice));
  memset(&g.dev, 0, sizeof(g.dev));
  g.dev.values = d;
  g.dev.n_nodes = (int32_t)nodes;
  const int32_t strides[3] = {dims[1] * dims[2], dims[2], 1};
  for (int a = 0; a < 3; ++a) {
    g.dev.dims[a] = dims[a];
    g.dev.stride[a] = dims[a] > 1 ? strides[a] : 0;
    g.dev.lo[a] = lo_log2[a];
    g.dev.scale[a] = dims[a] > 1 ? (float)((double)(dims[a] - 1) / ((double)hi_log2[a] - (double)lo_log2[a])) : 0.0f;
    // the measured hull on integers (density routing, Q16): ceil(2^lo) <= v <= floor(2^hi); a flat axis is unconstrained
    double vmin = dims[a] > 1 ? ceil(exp2((double)lo_log2[a])) : -2147483648.0;
    double vmax = dims[a] > 1 ? floor(exp2((double)hi_log2[a])) : 2147483647.0;
    if (dims[a] > 1 && vmin < 1.0) vmin = 1.0;                      // a non-positive axis value is outside
    g.dev.vmin[a] = (int32_t)fmax(vmin, -2147483648.0);
    g.dev.vmax[a] = (int32_t)fmin(vmax, 2147483647.0);
  }
  g.dev.route_idx = nullptr;
  g.dev.route_count = nullptr;
  memset(&g.tb, 0, sizeof(g.tb));
  g.tb.values = d;
  g.tb.bytes = (int32_t)(padded * 4);
  for (int a = 0; a < 3; ++a) {
    const bool flat = dims[a] <= 1;
    const double lo = flat ? 0.0 : (double)lo_log2[a];
    const double lor = nearbyint(lo);                    // the integer part of lo leaves with the exponent, exactly
    g.tb.stride4[a] = g.dev.stride[a] * 4;
    g.tb.nkc[a] = (float)-(8388608.0 + 127.0 + lor);
    g.tb.scale[a] = g.dev.scale[a];
    g.tb.nrs[a] = flat ? 0.0f : (float)(-(lo - lor) * (double)g.dev.scale[a]);
    g.tb.top[a] = (float)(dims[a] - 1);
    g.tb.vmin[a] = g.dev.vmin[a];
    g.tb.vmax[a] = g.dev.vmax[a];
  }
  g.values = d;
  g.loaded = true;
  return KS_OK;
}

}  // extern "C"

// =================================================================== compute entry points
namespace {

bool params_ok(const ks_step_params* p) {
  return p && isfinite(p->c_disp) && isfinite(p->floor_l) && isfinite(p->c_ovl) && isfinite(p->c_tail) &&
         isfinite(p->body_scale);
}

bool csr_ok(const int32_t* off, int n, long long limit) {       // host-resident CSR only
  if (off[0] < 0) return false;
  for (int i = 0; i < n; ++i)
    if (off[i + 1] < off[i]) return false;
  return limit < 0 || off[n] <= limit;
}

ks_status compose_device(ks_ctx* c, const float* const* lat, const int32_t* const* step_off, const int32_t* batch_n,
                         int n_batches, int n_steps, int n_specs, const ks_step_params* params,
                         const int32_t* cfg_off, int n_cfg, float* step_lat, float* cfg_lat,
                         const int32_t* const* mult = nullptr) {
  if (n_steps == 0 || n_specs == 0) {
    if (n_cfg > 0 && n_specs > 0) KS_CUDA(c, cudaMemsetAsync(cfg_lat, 0, (size_t)n_cfg * n_specs * 4, c->stream));
    return KS_OK;
  }
  KsComposeParams p;
  memset(&p, 0, sizeof(p));
  for (int b = 0; b < n_batches; ++b) {
    p.lat[b] = lat[b];
    p.step_off[b] = step_off[b];
    p.mult[b] = mult ? mult[b] : nullptr;
    p.spec_stride[b] = batch_n[b];
  }
  p.n_batches = n_batches;
  p.n_steps = n_steps;
  p.n_specs = n_specs;
  p.n_cfg = n_cfg;
  p.sp = *params;
  p.cfg_off = cfg_off;
  p.step_lat = step_lat;
  p.cfg_lat = cfg_lat;
  int launches = 0;
  KS_CUDA(c, ks_launch_compose(p, c->num_sms, c->stream, &launches));
  c->launches += launches;
  return KS_OK;
}

ks_status validate_compose(const ks_ctx* c, const float* const* lat, const int32_t* const* step_off,
                           const int32_t* batch_n, int n_batches, int n_steps, int n_specs,
                           const ks_step_params* params, const int32_t* cfg_off, int n_cfg, ks_mem_space space,
                           const float* step_lat, const float* cfg_lat, bool lat_optional,
                           const int32_t* const* mult = nullptr) {
  if (!c) return KS_EINVAL;
  if (space != KS_MEM_DEVICE && space != KS_MEM_HOST) return KS_EINVAL;
  if (n_batches < 0 || n_batches > KS_MAX_BATCHES || n_steps < 0 || n_specs < 0 || n_cfg < 0) return KS_EINVAL;
  if (!params_ok(params)) return KS_EINVAL;
  if (n_batches > 0 && (!step_off || !batch_n || (!lat && !lat_optional))) return KS_EINVAL;
  for (int b = 0; b < n_batches; ++b) {
    if (batch_n[b] < 0 || !step_off[b]) return KS_EINVAL;
    if (!lat_optional && !lat[b] && batch_n[b] > 0) return KS_EINVAL;
    // device space: the step kernel reads latencies (and multiplicities) with 16-byte loads
    if (space == KS_MEM_DEVICE && lat && lat[b] && !aligned16(lat[b])) return KS_EINVAL;
    if (space == KS_MEM_DEVICE && mult && mult[b] && !aligned16(mult[b])) return KS_EINVAL;
    if (space == KS_MEM_HOST && !csr_ok(step_off[b], n_steps, batch_n[b])) return KS_EINVAL;
  }
  if (n_cfg > 0 && (!cfg_off || !cfg_lat)) return KS_EINVAL;
  if (n_cfg > 0 && space == KS_MEM_HOST && !csr_ok(cfg_off, n_cfg, n_steps)) return KS_EINVAL;
  if ((long long)n_steps * n_specs > 0 && !step_lat) return KS_EINVAL;
  return KS_OK;
}

}  // namespace

extern "C" {

ks_status ks_predict_kernels(ks_ctx* c, const ks_desc_batch* batches, int n_batches, const ks_hw_spec* specs,
                             int n_specs, ks_tier tier, ks_mem_space space, float* const* latency,
                             int32_t* const* tiles, int32_t* const* waves, float* const* t_roof) {
  if (space != KS_MEM_DEVICE && space != KS_MEM_HOST) return KS_EINVAL;
  const bool dev = space == KS_MEM_DEVICE;
  ks_status st = validate_batches(c, batches, n_batches, specs, n_specs, tier, dev);
  if (st != KS_OK) return st;
  if (n_batches > 0 && !latency) return KS_EINVAL;
  for (int b = 0; b < n_batches; ++b) {
    if (batches[b].n == 0 || n_specs == 0) continue;
    if (!latency[b]) return KS_EINVAL;
    if (dev && (!aligned16(latency[b]) || (tiles && tiles[b] && !aligned16(tiles[b])) ||
                (waves && waves[b] && !aligned16(waves[b])) || (t_roof && t_roof[b] && !aligned16(t_roof[b]))))
      return KS_EINVAL;
  }
  if (c->sticky) return KS_ECUDA;
  if (n_batches == 0 || n_specs == 0) return KS_OK;
  KS_CUDA(c, cudaSetDevice(c->device));

  const void* cols[KS_MAX_BATCHES][KS_MAX_COLS] = {};
  DevOut outs[KS_MAX_BATCHES];
  if (dev) {
    for (int b = 0; b < n_batches; ++b) {
      for (int k = 0; k < batches[b].n_cols; ++k) cols[b][k] = batches[b].cols[k];
      outs[b].lat = latency[b];
      outs[b].tiles = tiles ? tiles[b] : nullptr;
      outs[b].waves = waves ? waves[b] : nullptr;
      outs[b].troof = t_roof ? t_roof[b] : nullptr;
    }
    RouteBuf rb[KS_MAX_BATCHES];
    if (tier == KS_TIER_B_ROUTED) {                  // the row lists live in the library workspace (stream-ordered reuse)
      st = ws_reserve(c, route_need(batches, n_batches, tier));
      if (st != KS_OK) return st;
      route_take(c, batches, n_batches, tier, rb);
    }
    return predict_device(c, batches, cols, n_batches, specs, n_specs, tier, outs, rb);
  }
  // host space: stage through the workspace
  size_t need = 0;
  for (int b = 0; b < n_batches; ++b) {
    const size_t n = batches[b].n, o = align_up(n * (size_t)n_specs * 4, 256);
    need += batches[b].n_cols * align_up(n * 4, 256) + o;
    if (tiles && tiles[b]) need += o;
    if (waves && waves[b]) need += o;
    if (t_roof && t_roof[b]) need += o;
  }
  need += route_need(batches, n_batches, tier);
  st = ws_reserve(c, need);
  if (st != KS_OK) return st;
  RouteBuf rb[KS_MAX_BATCHES];
  route_take(c, batches, n_batches, tier, rb);
  for (int b = 0; b < n_batches; ++b) {
    const size_t n = batches[b].n, ob = n * (size_t)n_specs * 4;
    for (int k = 0; k < batches[b].n_cols; ++k) {
      void* d = ws_take(c, n * 4);
      if (n) KS_CUDA(c, cudaMemcpyAsync(d, batches[b].cols[k], n * 4, cudaMemcpyHostToDevice, c->stream));
      cols[b][k] = d;
    }
    outs[b].lat = static_cast<float*>(ws_take(c, ob));
    if (tiles && tiles[b]) outs[b].tiles = static_cast<int32_t*>(ws_take(c, ob));
    if (waves && waves[b]) outs[b].waves = static_cast<int32_t*>(ws_take(c, ob));
    if (t_roof && t_roof[b]) outs[b].troof = static_cast<float*>(ws_take(c, ob));
  }
  st = predict_device(c, batches, cols, n_batches, specs, n_specs, tier, outs, rb);
  if (st != KS_OK) return st;
  for (int b = 0; b < n_batches; ++b) {
    const size_t ob = (size_t)batches[b].n * n_specs * 4;
    if (!ob) continue;
    KS_CUDA(c, cudaMemcpyAsync(latency[b], outs[b].lat, ob, cudaMemcpyDeviceToHost, c->stream));
    if (outs[b].tiles) KS_CUDA(c, cudaMemcpyAsync(tiles[b], outs[b].tiles, ob, cudaMemcpyDeviceToHost, c->stream));
    if (outs[b].waves) KS_CUDA(c, cudaMemcpyAsync(waves[b], outs[b].waves, ob, cudaMemcpyDeviceToHost, c->stream));
    if (outs[b].troof) KS_CUDA(c, cudaMemcpyAsync(t_roof[b], outs[b].troof, ob, cudaMemcpyDeviceToHost, c->stream));
  }
  KS_CUDA(c, cudaStreamSynchronize(c->stream));
  return KS_OK;
}

}  // extern "C"

// ---- ks_predict_routed_static (include/ks.h): density routing with its row lists in a fixed device array.
// Per routed bucket the lists take align_up(4 n, 256) + 256 bytes (route_need), at most 4 n + 511: the array holds
// KS_STATIC_ROUTE_MAX_ROWS rows in up to KS_MAX_BATCHES buckets.  Every GPU that loads libks holds it until exit.
// In host code `ks_static_route` is a host-side stand-in, not a device address: the kernels get the pointer that
// cudaGetSymbolAddress returns, resolved once per device with that device current.
namespace {

constexpr size_t kStaticRouteBytes = (size_t)KS_STATIC_ROUTE_MAX_ROWS * 4 + (size_t)KS_MAX_BATCHES * 512;
constexpr int kStaticMaxDevices = 64;

}  // namespace

static __device__ __align__(256) unsigned char ks_static_route[kStaticRouteBytes];

namespace {

std::mutex g_static_mu;
unsigned char* g_static_ptr[kStaticMaxDevices] = {};

// the array's address on the CURRENT device (the caller has made c->device current)
ks_status static_route_ptr(ks_ctx* c, unsigned char** out) {
  if (c->device < 0 || c->device >= kStaticMaxDevices) return KS_EUNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[c->device]) {
    void* p = nullptr;
    KS_CUDA(c, cudaGetSymbolAddress(&p, ks_static_route));
    if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return cuda_fail(c);
    g_static_ptr[c->device] = static_cast<unsigned char*>(p);
  }
  *out = g_static_ptr[c->device];
  return KS_OK;
}

}  // namespace

extern "C" {

ks_status ks_predict_routed_static(ks_ctx* c, const ks_desc_batch* batches, int n_batches, const ks_hw_spec* specs,
                                   int n_specs, float* const* latency, int32_t* const* tiles, int32_t* const* waves,
                                   float* const* t_roof) {
  const int tier = KS_TIER_B_ROUTED;
  ks_status st = validate_batches(c, batches, n_batches, specs, n_specs, tier, true);
  if (st != KS_OK) return st;
  if (n_batches > 0 && !latency) return KS_EINVAL;
  long long rows = 0;
  for (int b = 0; b < n_batches; ++b) {
    if (batches[b].family != KS_FAM_ALLREDUCE) rows += batches[b].n;
    if (batches[b].n == 0 || n_specs == 0) continue;
    if (!latency[b]) return KS_EINVAL;
    if (!aligned16(latency[b]) || (tiles && tiles[b] && !aligned16(tiles[b])) ||
        (waves && waves[b] && !aligned16(waves[b])) || (t_roof && t_roof[b] && !aligned16(t_roof[b])))
      return KS_EINVAL;
  }
  if (rows > (long long)KS_STATIC_ROUTE_MAX_ROWS) return KS_ELIMIT;        // the fixed array holds no more
  if (route_need(batches, n_batches, tier) > kStaticRouteBytes) return KS_ELIMIT;
  if (c->sticky) return KS_ECUDA;
  if (n_batches == 0 || n_specs == 0) return KS_OK;
  KS_CUDA(c, cudaSetDevice(c->device));
  unsigned char* base = nullptr;
  st = static_route_ptr(c, &base);
  if (st != KS_OK) return st;

  const void* cols[KS_MAX_BATCHES][KS_MAX_COLS] = {};
  DevOut outs[KS_MAX_BATCHES];
  RouteBuf rb[KS_MAX_BATCHES];
  size_t used = 0;
  for (int b = 0; b < n_batches; ++b) {
    for (int k = 0; k < batches[b].n_cols; ++k) cols[b][k] = batches[b].cols[k];
    outs[b].lat = latency[b];
    outs[b].tiles = tiles ? tiles[b] : nullptr;
    outs[b].waves = waves ? waves[b] : nullptr;
    outs[b].troof = t_roof ? t_roof[b] : nullptr;
    if (batches[b].family == KS_FAM_ALLREDUCE) continue;
    rb[b].idx = reinterpret_cast<int32_t*>(base + used);
    used += align_up((size_t)batches[b].n * 4, 256);
    rb[b].count = reinterpret_cast<int32_t*>(base + used);   // cleared (stream-ordered) by predict_device before pass 1
    used += 256;
  }
  return predict_device(c, batches, cols, n_batches, specs, n_specs, tier, outs, rb);
}

ks_status ks_compose_steps(ks_ctx* c, const float* const* latency, const int32_t* const* step_off,
                           const int32_t* batch_n, int n_batches, int n_steps, int n_specs,
                           const ks_step_params* params, const int32_t* cfg_off, int n_cfg, ks_mem_space space,
                           float* step_latency, float* cfg_latency) {
  return ks_compose_steps_weighted(c, latency, nullptr, step_off, batch_n, n_batches, n_steps, n_specs, params, cfg_off,
                                   n_cfg, space, step_latency, cfg_latency);
}

ks_status ks_compose_steps_weighted(ks_ctx* c, const float* const* latency, const int32_t* const* mult,
                                    const int32_t* const* step_off, const int32_t* batch_n, int n_batches,
                                    int n_steps, int n_specs, const ks_step_params* params, const int32_t* cfg_off,
                                    int n_cfg, ks_mem_space space, float* step_latency, float* cfg_latency) {
  ks_status st = validate_compose(c, latency, step_off, batch_n, n_batches, n_steps, n_specs, params, cfg_off, n_cfg,
                                  space, step_latency, cfg_latency, false, mult);
  if (st != KS_OK) return st;
  if (c->sticky) return KS_ECUDA;
  KS_CUDA(c, cudaSetDevice(c->device));
  if (space == KS_MEM_DEVICE)
    return compose_device(c, latency, step_off, batch_n, n_batches, n_steps, n_specs, params, cfg_off, n_cfg,
                          step_latency, cfg_latency, mult);
  size_t need = align_up((size_t)(n_cfg + 1) * 4, 256) + align_up((size_t)n_steps * n_specs * 4, 256) +
                align_up((size_t)n_cfg * n_specs * 4 + 4, 256);
  for (int b = 0; b < n_batches; ++b)
    need += align_up((size_t)batch_n[b] * n_specs * 4, 256) + align_up((size_t)(n_steps + 1) * 4, 256) +
            align_up((size_t)batch_n[b] * 4, 256);
  st = ws_reserve(c, need);
  if (st != KS_OK) return st;
  const float* dlat[KS_MAX_BATCHES];
  const int32_t* doff[KS_MAX_BATCHES];
  const int32_t* dmult[KS_MAX_BATCHES] = {};
  for (int b = 0; b < n_batches; ++b) {
    if (mult && mult[b] && batch_n[b] > 0) {
      int32_t* dm = static_cast<int32_t*>(ws_take(c, (size_t)batch_n[b] * 4));
      KS_CUDA(c, cudaMemcpyAsync(dm, mult[b], (size_t)batch_n[b] * 4, cudaMemcpyHostToDevice, c->stream));
      dmult[b] = dm;
    }
    const size_t lb = (size_t)batch_n[b] * n_specs * 4, ob = (size_t)(n_steps + 1) * 4;
    float* dl = static_cast<float*>(ws_take(c, lb));
    int32_t* dofs = static_cast<int32_t*>(ws_take(c, ob));
    if (lb) KS_CUDA(c, cudaMemcpyAsync(dl, latency[b], lb, cudaMemcpyHostToDevice, c->stream));
    KS_CUDA(c, cudaMemcpyAsync(dofs, step_off[b], ob, cudaMemcpyHostToDevice, c->stream));
    dlat[b] = dl;
    doff[b] = dofs;
  }
  int32_t* dcfg = static_cast<int32_t*>(ws_take(c, (size_t)(n_cfg + 1) * 4));
  float* dstep = static_cast<float*>(ws_take(c, (size_t)n_steps * n_specs * 4));
  float* dtot = static_cast<float*>(ws_take(c, (size_t)n_cfg * n_specs * 4 + 4));
  if (n_cfg > 0) KS_CUDA(c, cudaMemcpyAsync(dcfg, cfg_off, (size_t)(n_cfg + 1) * 4, cudaMemcpyHostToDevice, c->stream));
  st = compose_device(c, dlat, doff, batch_n, n_batches, n_steps, n_specs, params, dcfg, n_cfg, dstep, dtot, dmult);
  if (st != KS_OK) return st;
  if ((size_t)n_steps * n_specs)
    KS_CUDA(c, cudaMemcpyAsync(step_latency, dstep, (size_t)n_steps * n_specs * 4, cudaMemcpyDeviceToHost, c->stream));
  if ((size_t)n_cfg * n_specs)
    KS_CUDA(c, cudaMemcpyAsync(cfg_latency, dtot, (size_t)n_cfg * n_specs * 4, cudaMemcpyDeviceToHost, c->stream));
  KS_CUDA(c, cudaStreamSynchronize(c->stream));
  return KS_OK;
}

ks_status ks_run_steps(ks_ctx* c, const ks_desc_batch* batches, const int32_t* const* step_off, int n_batches,
                       const ks_hw_spec* specs, int n_specs, ks_tier tier, int n_steps, const ks_step_params* params,
                       const int32_t* cfg_off, int n_cfg, ks_mem_space space, float* const* latency,
                       float* step_latency, float* cfg_latency) {
  if (space != KS_MEM_DEVICE && space != KS_MEM_HOST) return KS_EINVAL;
  const bool dev = space == KS_MEM_DEVICE;
  ks_status st = validate_batches(c, batches, n_batches, specs, n_specs, tier, dev);
  if (st != KS_OK) return st;
  int32_t batch_n[KS_MAX_BATCHES] = {0};
  for (int b = 0; b < n_batches; ++b) batch_n[b] = batches[b].n;
  st = validate_compose(c, latency, step_off, batch_n, n_batches, n_steps, n_specs, params, cfg_off, n_cfg, space,
                        step_latency, cfg_latency, true);
  if (st != KS_OK) return st;
  if (dev)
    for (int b = 0; b < n_batches; ++b)
      if ((latency && latency[b] && !aligned16(latency[b])) || (batches[b].mult && !aligned16(batches[b].mult)))
        return KS_EINVAL;
  if (c->sticky) return KS_ECUDA;
  KS_CUDA(c, cudaSetDevice(c->device));

  // Tier NONE with one spec vector (config 4a's shape; also the closed loop's weighted rows): ONE kernel computes the latencies in
  // the step kernel's staging phase (ks_fused.cu) instead of writing them to HBM and reading them back; per-kernel
  // latencies are written only where the caller passed a buffer.  Same bits as the two-call path.
  if (dev && tier == KS_TIER_NONE && n_specs == 1 && n_steps > 0 && n_batches >= 1 && n_batches <= KS_FUSED_MAX_BUCKETS) {
    bool fusable = true, weighted = false;
    long long rows = 0;
    for (int b = 0; b < n_batches; ++b) {
      fusable = fusable && ks_fused_none_supported(batches[b].family, batches[b].col_dtype == KS_COL_F32);
      weighted = weighted || batches[b].mult != nullptr;
      rows += batches[b].n;
    }
    // an average chunk of 32 steps must fit the staging buffer (a chunk that does not is summed from the columns)
    fusable = fusable && (double)rows / (double)n_steps * 32.0 <= 0.85 * (double)ks_fused_none_cap_floats(weighted);
    if (fusable) {
      KsFusedParams p;
      memset(&p, 0, sizeof(p));
      for (int b = 0; b < n_batches; ++b) {
        DevOut o;
        o.lat = latency ? latency[b] : nullptr;
        p.bk[b] = make_bucket_dev(batches[b], batches[b].cols, o, 0);
        p.step_off[b] = step_off[b];
        p.mult[b] = batches[b].mult;
      }
      p.n_batches = n_batches;
      p.n_steps = n_steps;
      p.sp = *params;
      p.spec = make_spec_dev(specs[0]);
      p.step_lat = step_latency;
      KS_CUDA(c, ks_launch_fused_none(p, c->stream));
      c->launches += 1;
      KsComposeParams q;
      memset(&q, 0, sizeof(q));
      q.n_steps = n_steps;
      q.n_specs = 1;
      q.n_cfg = n_cfg;
      q.cfg_off = cfg_off;
      q.step_lat = step_latency;
      q.cfg_lat = cfg_latency;
      int launches = 0;
      KS_CUDA(c, ks_launch_cfg_totals(q, c->stream, true, &launches));
      c->launches += launches;
      return KS_OK;
    }
  }

  size_t need = 0;
  for (int b = 0; b < n_batches; ++b) {
    const size_t n = batches[b].n;
    const bool user_lat = dev && latency && latency[b];
    if (!user_lat) need += align_up(n * (size_t)n_specs * 4, 256);
    if (!dev) need += (batches[b].n_cols + 1) * align_up(n * 4, 256) + align_up((size_t)(n_steps + 1) * 4, 256);
  }
  if (!dev)
    need += align_up((size_t)(n_cfg + 1) * 4, 256) + align_up((size_t)n_steps * n_specs * 4, 256) +
            align_up((size_t)n_cfg * n_specs * 4 + 4, 256);
  need += route_need(batches, n_batches, tier);
  st = ws_reserve(c, need);
  if (st != KS_OK) return st;
  RouteBuf rb[KS_MAX_BATCHES];
  route_take(c, batches, n_batches, tier, rb);

  const void* cols[KS_MAX_BATCHES][KS_MAX_COLS] = {};
  DevOut outs[KS_MAX_BATCHES];
  const float* dlat[KS_MAX_BATCHES];
  const int32_t* doff[KS_MAX_BATCHES];
  const int32_t* dmult[KS_MAX_BATCHES] = {};       // layer-homogeneous multiplicities, optional
  if (dev) {
    for (int b = 0; b < n_batches; ++b) {
      for (int k = 0; k < batches[b].n_cols; ++k) cols[b][k] = batches[b].cols[k];
      outs[b].lat = (latency && latency[b]) ? latency[b]
                                            : static_cast<float*>(ws_take(c, (size_t)batches[b].n * n_specs * 4));
      dlat[b] = outs[b].lat;
      doff[b] = step_off[b];
      dmult[b] = batches[b].mult;
    }
    if (n_specs > 0 && n_batches > 0) {
      st = predict_device(c, batches, cols, n_batches, specs, n_specs, tier, outs, rb);
      if (st != KS_OK) return st;
    }
    return compose_device(c, dlat, doff, batch_n, n_batches, n_steps, n_specs, params, cfg_off, n_cfg, step_latency,
                          cfg_latency, dmult);
  }

  // ---- host space: a three-stream pipeline over the buckets (largest copy first is the caller's
  // order).  h2d: columns + offsets of bucket b; stream: predict bucket b as soon as its inputs have
  // landed; d2h: bucket b's latencies go back while bucket b+1 is predicted.  Composition and the
  // small step/config results stay on the ctx stream.  Ends with a synchronisation of both.
  st = pipeline_init(c);
  if (st != KS_OK) return st;
  KS_CUDA(c, cudaEventRecord(c->ev_start, c->stream));            // earlier work on the ctx stream owns the workspace
  KS_CUDA(c, cudaStreamWaitEvent(c->h2d, c->ev_start, 0));
  for (int b = 0; b < n_batches; ++b) {
    const size_t n = batches[b].n;
    // columns that lie back to back in host memory (one block per bucket) move with ONE copy: a step is
    // PCIe-bound and every separate copy costs a few microseconds of link idle time
    bool adjacent = n > 0 && n % 4 == 0 && batches[b].n_cols > 1;
    for (int k = 0; adjacent && k + 1 < batches[b].n_cols; ++k)
      adjacent = static_cast<const char*>(batches[b].cols[k + 1]) == static_cast<const char*>(batches[b].cols[k]) + n * 4;
    if (adjacent) {
      char* d = static_cast<char*>(ws_take(c, n * 4 * batches[b].n_cols));
      KS_CUDA(c, cudaMemcpyAsync(d, batches[b].cols[0], n * 4 * batches[b].n_cols, cudaMemcpyHostToDevice, c->h2d));
      for (int k = 0; k < batches[b].n_cols; ++k) cols[b][k] = d + (size_t)k * n * 4;
    } else {
      for (int k = 0; k < batches[b].n_cols; ++k) {
        void* d = ws_take(c, n * 4);
        if (n) KS_CUDA(c, cudaMemcpyAsync(d, batches[b].cols[k], n * 4, cudaMemcpyHostToDevice, c->h2d));
        cols[b][k] = d;
      }
    }
    int32_t* dofs = static_cast<int32_t*>(ws_take(c, (size_t)(n_steps + 1) * 4));
    KS_CUDA(c, cudaMemcpyAsync(dofs, step_off[b], (size_t)(n_steps + 1) * 4, cudaMemcpyHostToDevice, c->h2d));
    doff[b] = dofs;
    if (batches[b].mult && n) {
      int32_t* dm = static_cast<int32_t*>(ws_take(c, n * 4));
      KS_CUDA(c, cudaMemcpyAsync(dm, batches[b].mult, n * 4, cudaMemcpyHostToDevice, c->h2d));
      dmult[b] = dm;
    }
    outs[b].lat = static_cast<float*>(ws_take(c, n * (size_t)n_specs * 4));
    dlat[b] = outs[b].lat;
    KS_CUDA(c, cudaEventRecord(c->ev_in[b], c->h2d));
  }
  int32_t* dcfg = static_cast<int32_t*>(ws_take(c, (size_t)(n_cfg + 1) * 4));
  if (n_cfg > 0) KS_CUDA(c, cudaMemcpyAsync(dcfg, cfg_off, (size_t)(n_cfg + 1) * 4, cudaMemcpyHostToDevice, c->h2d));
  KS_CUDA(c, cudaEventRecord(c->ev_start, c->h2d));
  float* dstep = static_cast<float*>(ws_take(c, (size_t)n_steps * n_specs * 4));
  float* dtot = static_cast<float*>(ws_take(c, (size_t)n_cfg * n_specs * 4 + 4));
  for (int b = 0; b < n_batches; ++b) {
    KS_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_in[b], 0));
    if (n_specs > 0 && batches[b].n > 0) {
      st = predict_device(c, batches + b, cols + b, 1, specs, n_specs, tier, outs + b, rb + b);
      if (st != KS_OK) return st;
    }
    const size_t ob = (size_t)batches[b].n * n_specs * 4;
    if (latency && latency[b] && ob) {
      KS_CUDA(c, cudaEventRecord(c->ev_out[b], c->stream));
      KS_CUDA(c, cudaStreamWaitEvent(c->d2h, c->ev_out[b], 0));
      KS_CUDA(c, cudaMemcpyAsync(latency[b], outs[b].lat, ob, cudaMemcpyDeviceToHost, c->d2h));
    }
  }
  KS_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_start, 0));     // cfg offsets (and every earlier h2d copy)
  st = compose_device(c, dlat, doff, batch_n, n_batches, n_steps, n_specs, params, dcfg, n_cfg, dstep, dtot, dmult);
  if (st != KS_OK) return st;
  if ((size_t)n_steps * n_specs)
    KS_CUDA(c, cudaMemcpyAsync(step_latency, dstep, (size_t)n_steps * n_specs * 4, cudaMemcpyDeviceToHost, c->stream));
  if ((size_t)n_cfg * n_specs)
    KS_CUDA(c, cudaMemcpyAsync(cfg_latency, dtot, (size_t)n_cfg * n_specs * 4, cudaMemcpyDeviceToHost, c->stream));
  KS_CUDA(c, cudaStreamSynchronize(c->stream));
  KS_CUDA(c, cudaStreamSynchronize(c->d2h));
  return KS_OK;
}

}  // extern "C"
