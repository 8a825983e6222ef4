// ks_mlp_common.cuh — pieces shared by the two Tier-A kernels (ks_mlp_ws.cu: H <= 128; ks_mlp_ws256.cu:
// H = 256; both warp-specialized tcgen05 pipelines; ks_mlp.cu picks one by head width).
#pragma once
#include "ks_internal.h"
#include "ks_ptx.cuh"

namespace ksmlp {

template <int FAM> struct NCols { static constexpr int v = 3; };
template <> struct NCols<KS_FAM_GROUPED_GEMM> { static constexpr int v = 10; };
template <> struct NCols<KS_FAM_ELEMWISE> { static constexpr int v = 2; };

constexpr int kRows = 128;                 // rows per tile = TMEM lanes
constexpr int kChunkBytes = kRows * 16;    // one K chunk (8 bf16) of a 128-row operand

// Hidden activation, scaled by two: g2(x) = 2 GELU(x) = x + x tanh(sqrt(2/pi) (x + 0.044715 x^3)).
// The factor 1/2 is folded into the next layer's weights at ks_load_heads (exact in bf16), which
// saves one multiply per activation.  4 FMA-pipe instructions + 1 MUFU.TANH.
KS_PTX float gelu2_f32(float x) {
  const float x2 = x * x;
  const float p = fmaf(x2, 0.0356774081f, 0.7978845608f);
  const float t = ks_tanh_approx(x * p);
  return fmaf(x, t, x);
}
// Two activations at once with packed fp32 instructions (FMUL2, FFMA2, FMUL2, 2 x MUFU.TANH, FFMA2):
// bit-identical to gelu2_f32 on each element, 3 issue slots per activation instead of 5.
KS_PTX void gelu2_f32x2(float xa, float xb, float& ga, float& gb) {
  float x2a, x2b, pa, pb, ua, ub;
  ks_mul2(x2a, x2b, xa, xb, xa, xb);
  ks_fma2(pa, pb, x2a, x2b, 0.0356774081f, 0.0356774081f, 0.7978845608f, 0.7978845608f);
  ks_mul2(ua, ub, xa, xb, pa, pb);
  const float ta = ks_tanh_approx(ua), tb = ks_tanh_approx(ub);
  ks_fma2(ga, gb, xa, xb, ta, tb, xa, xb);
}
// packed bf16x2 variant (two activations per FMA-pipe instruction; MUFU.TANH.BF16 per half)
KS_PTX uint32_t gelu2_bf16x2(float a, float b) {
  const uint32_t x = ks_pack_bf16x2(a, b);
  const uint32_t x2 = ks_mul_bf16x2(x, x);
  const uint32_t p = ks_fma_bf16x2(x2, 0x3D123D12u /*0.0356*/, 0x3F4C3F4Cu /*0.7969*/);
  const uint32_t t = ks_tanh_bf16x2(ks_mul_bf16x2(x, p));
  return ks_fma_bf16x2(x, t, x);
}

// Decode + roofline + features of one descriptor row for one spec; packs the bf16 A1 row
// (K1 values, bias columns set to 1) into q[K1/8] and returns t_roof.  S1-S3 of DESIGN.md.
template <int FAM, int NIN, int K1, int BIAS_ROW>
KS_DEV float feature_row(const int* v, const KsBucketDev& bk, const KsSpecDev& sp, uint4* q, KsWork& w, KsRoof& rf) {
  w = ks_decode<FAM>(v, bk, sp);
  rf = ks_roofline(w, sp);
  float x[K1];
  ks_features<FAM, (NIN == 32 ? 22 : NIN)>(v, bk, sp, w, rf, x);
#pragma unroll
  for (int i = (NIN == 32 ? 22 : NIN); i < K1; ++i) x[i] = 0.0f;
  x[BIAS_ROW] = 1.0f;          // multiplies the b1_hi row of the W1 image
  x[BIAS_ROW + 1] = 1.0f;      // multiplies the b1_lo row
#pragma unroll
  for (int kc = 0; kc < K1 / 8; ++kc) {
    q[kc].x = ks_pack_bf16x2(x[kc * 8 + 0], x[kc * 8 + 1]);
    q[kc].y = ks_pack_bf16x2(x[kc * 8 + 2], x[kc * 8 + 3]);
    q[kc].z = ks_pack_bf16x2(x[kc * 8 + 4], x[kc * 8 + 5]);
    q[kc].w = ks_pack_bf16x2(x[kc * 8 + 6], x[kc * 8 + 7]);
  }
  return rf.t_roof;
}

// Tile bookkeeping of a launch, computed in the kernel: a bucket may be a row LIST whose length is
// only known on the device (density routing: idx[0 .. *count)), so the tile prefix cannot come from
// the host.  ne[b] = rows (or list entries) of bucket b, tb[b] = first 128-row tile of bucket b.
struct TileMap {
  int tb[KS_MLP_MAX_BUCKETS + 1];
  int ne[KS_MLP_MAX_BUCKETS];
};
KS_DEV void tile_map_init(const KsMlpParams& p, TileMap* tm) {   // one thread
  int t = 0;
  for (int b = 0; b < p.n_buckets; ++b) {
    int n = p.bk[b].n;
    if (p.bk[b].count) { const int c = __ldg(p.bk[b].count); n = c < n ? c : n; }
    tm->ne[b] = n;
    tm->tb[b] = t;
    t += (n + kRows - 1) / kRows;
  }
  for (int b = p.n_buckets; b <= KS_MLP_MAX_BUCKETS; ++b) tm->tb[b] = t;
}
// position i of a bucket -> descriptor row (identity unless the bucket is a row list)
KS_DEV int map_row(const KsBucketDev& bk, int i) { return bk.idx ? __ldg(bk.idx + i) : i; }

// raw 32-bit column load (int32 or fp32 bits); converted at the point of use so a prefetch does
// not stall on the conversion
KS_DEV int load_col_raw(const void* col, int i) { return __ldg((const int*)col + i); }
KS_DEV int col_value(int raw, bool f32) { return f32 ? __float2int_rn(__int_as_float(raw)) : raw; }

}  // namespace ksmlp
