// ks_internal.h — launcher interfaces between the C-ABI layer (ks_api.cu) and the kernels.
#pragma once
#include "ks_common.cuh"

struct KsSpecTable {
  KsSpecDev s[KS_MAX_SPECS_PER_LAUNCH];
};

// ---- streaming kernels (Tier NONE / Tier B): ks_stream.cu
#define KS_TIER_BOUNDED 100  // internal: Tier A with the bounded analytical head (streaming kernel)
#define KS_BOUNDED_NF 22    // real features of the largest feature vector (Q2: 22..31 are zero)
struct KsBoundedDev {
  float w_gamma[KS_BOUNDED_NF], w_alpha[KS_BOUNDED_NF];   // zero beyond the head's n_in
  float b_gamma, b_alpha;
};
struct KsStreamParams {
  KsBucketDev bk;
  KsGridDev grid;          // Tier B only
  KsBoundedDev bounded;    // KS_TIER_BOUNDED only
  int32_t n_specs;
  int32_t tier;
  int64_t spec_stride;     // elements between consecutive specs in the outputs (= bucket n)
  KsSpecTable specs;
};
cudaError_t ks_launch_stream(const KsStreamParams& p, int num_sms, cudaStream_t st);

// ---- Tier B, GEMM and attention families, all buckets of a call in one persistent launch: ks_tierb.cu
#define KS_TIERB_MAX_BUCKETS 4
struct KsTierBGrid {
  const float* values;     // device; `bytes` bytes (a multiple of 16): the nodes, then stride[0] + stride[1] + 2 zero floats
                           // (the corners one node past the last node are read with weight 0)
  int32_t bytes;
  int32_t stride4[3];      // byte strides; 0 for a flat (1-node) axis
  float nkc[3];            // -(2^23 + 127 + round(lo)): (2^23 + biased exponent) + nkc is exact
  float nrs[3];            // -(lo - round(lo)) * scale: the remainder of lo, folded into the coordinate's FMA
  float scale[3];          // (dims-1)/(hi-lo); 0 for a flat axis
  float top[3];            // dims - 1
  int32_t vmin[3], vmax[3];   // the hull on integers (Q16)
  int32_t* route_idx;      // KS_TIER_B_ROUTED pass 1 (nullptr = plain Tier B)
  int32_t* route_count;
};
struct KsTierBParams {
  KsBucketDev bk[KS_TIERB_MAX_BUCKETS];
  KsTierBGrid grid[KS_TIERB_MAX_BUCKETS];
  int32_t tile_begin[KS_TIERB_MAX_BUCKETS + 1];   // filled by the launcher: prefix of the buckets' 4-row x NT tiles
  int32_t cta_begin[KS_TIERB_MAX_BUCKETS + 1];    // ... and of the CTAs that serve them
  int32_t n_buckets, n_specs, pad;
  KsSpecTable specs;
};
cudaError_t ks_launch_tierb(const KsTierBParams& p, int num_sms, cudaStream_t st);

// Small Tier-NONE calls (the closed simulation loop prices a few thousand rows per pass): all buckets in
// ONE launch, a thread per row.  Same per-row device functions as the streaming kernel, so the same bits.
#define KS_STREAM_SMALL_MAX_ROWS 32768
struct KsStreamSmallParams {
  KsBucketDev bk[KS_MAX_BATCHES];
  int32_t row_begin[KS_MAX_BATCHES + 1];   // prefix of the buckets' row counts
  int32_t n_buckets, n_specs, pad;
  KsSpecTable specs;
};
cudaError_t ks_launch_stream_small(const KsStreamSmallParams& p, cudaStream_t st);

// ---- Tier-A MLP head kernel: ks_mlp.cu
#define KS_MLP_MAX_BUCKETS 4
struct KsHeadDev {
  const void* w1_img;      // bf16 UMMA image [K1/8][H][8]  (rows n_in, n_in+1 hold b1 hi/lo)
  const void* w2_img;      // bf16 UMMA image [(H+24)/8][H][8] (K rows H, H+1 hold b2 hi/lo; the last K chunk holds them again at
                           // the chunk positions of layer 1's constant-1 columns: the H = 256 kernel's bias MMA, ks_mlp_ws256.cu)
  const float* w3;         // fp32 [H], holds w3 / 2
  const float* b2;         // fp32 [H] (the H = 256 kernel adds b2 in its fp32 epilogue)
  float b3;
  int32_t members;         // > 1: MLP ensemble (Q17) of `members` heads, H / members columns each:
                           // W1/b1/b2/w3 concatenated, W2 block-diagonal, one output bias per member
  float b3m[KS_MAX_ENSEMBLE];
  // single MLP head: eta = out_add + exp(max(out_sgn * z, out_lo)), i.e. 1 + exp(-z) for a utilisation output
  // (-1, -inf, 1) or exp(max(z, 0)) for a log-eta output (+1, 0, 0); ks_set_head_output
  float out_sgn, out_lo, out_add;
};
struct KsMlpParams {
  KsBucketDev bk[KS_MLP_MAX_BUCKETS];
  KsHeadDev head[KS_MLP_MAX_BUCKETS];
  int32_t tile_begin[KS_MLP_MAX_BUCKETS + 1];   // prefix of 128-row tiles per bucket
  int32_t n_buckets, n_specs, gelu_mode, any_ens;   // any_ens: some head of the launch is an ensemble
  KsSpecTable specs;
};
// n_in in {8,12,32}; h in {64,128,256}; all buckets of one launch share (n_in, h)
cudaError_t ks_launch_mlp(const KsMlpParams& p, int n_in, int h, int num_sms, cudaStream_t st);
cudaError_t ks_launch_mlp_ws(const KsMlpParams& p, int n_in, int h, int num_sms, cudaStream_t st);   // h <= 128
cudaError_t ks_launch_mlp_ws256(const KsMlpParams& p, int n_in, int num_sms, cudaStream_t st);            // h == 256
// sizes of the device weight images for a head
size_t ks_mlp_w1_img_bytes(int n_in, int h);
size_t ks_mlp_w2_img_bytes(int h);
int ks_mlp_k1(int n_in);   // padded K of layer 1 (16 or 32)

// ---- step composition: ks_compose.cu
struct KsComposeParams {
  const float* lat[KS_MAX_BATCHES];
  const int32_t* step_off[KS_MAX_BATCHES];
  const int32_t* mult[KS_MAX_BATCHES];    // optional per-row multiplicities (nullptr = ones)
  int64_t spec_stride[KS_MAX_BATCHES];
  int32_t n_batches, n_steps, n_specs, n_cfg;
  int32_t cap_floats;                     // staging buffer of a CTA in floats (set by the launcher)
  ks_step_params sp;
  const int32_t* cfg_off;
  float* step_lat;   // [n_specs][n_steps]
  float* cfg_lat;    // [n_specs][n_cfg]
};
// for ks_sched.cu (the simulation loop lives outside ks_api.cu): the context's stream and device
cudaStream_t ks_internal_stream(ks_ctx* c);
cudaError_t ks_internal_set_device(ks_ctx* c);
cudaError_t ks_launch_compose(const KsComposeParams& p, int num_sms, cudaStream_t st, int* launches);
// S7's second half alone (per-configuration totals of p.step_lat); after_ours: the launch may overlap the tail of
// the libks kernel that precedes it on the stream (it waits for that kernel's completion itself)
cudaError_t ks_launch_cfg_totals(const KsComposeParams& p, cudaStream_t st, bool after_ours, int* launches);

// ---- Tier NONE, one spec, unweighted: decode + roofline + floor + step sums + Eq. 4 in one kernel: ks_fused.cu
#define KS_FUSED_MAX_BUCKETS 8
struct KsFusedParams {
  KsBucketDev bk[KS_FUSED_MAX_BUCKETS];      // lat may be nullptr: the per-kernel latencies are not written then
  const int32_t* step_off[KS_FUSED_MAX_BUCKETS];
  const int32_t* mult[KS_FUSED_MAX_BUCKETS];  // optional per-row multiplicities (nullptr = ones)
  int32_t n_batches, n_steps, cap_floats, pad;
  ks_step_params sp;
  KsSpecDev spec;
  float* step_lat;                           // [n_steps]
};
bool ks_fused_none_supported(int family, bool col_f32);
cudaError_t ks_launch_fused_none(const KsFusedParams& p, cudaStream_t st);
int ks_fused_none_cap_floats(bool weighted);   // staging capacity of a chunk (floats)

// Every libks kernel is launched with programmatic stream serialization and opens with
//   griddepcontrol.launch_dependents;  cudaGridDependencySynchronize();
// so its launch latency and CTA scheduling overlap the tail of whatever kernel precedes it on the stream, while
// nothing is read or written before that kernel has completed and flushed (the same ordering as a plain launch).
template <typename Kern, typename Params>
inline cudaError_t ks_launch_pdl(Kern kern, unsigned blocks, unsigned threads, size_t smem, cudaStream_t st, const Params& p) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(blocks);
  cfg.blockDim = dim3(threads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, p);
}
