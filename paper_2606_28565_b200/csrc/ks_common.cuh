// ks_common.cuh — device-side building blocks shared by the libks kernels (sm_100a only).
// S1 descriptor decode (F_comp, F_mem, B), S2 roofline + wave quantization (Eq. 2,
// PAPER.md:88 Fig. 2), S3 dimensionless features (Q2).  fp32 arithmetic,
// exact integer tile/wave math.  No code is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/ks.h"

#define KS_DEV __device__ __forceinline__

// ------------------------------------------------------------------ exact division by an invariant
// q = floor(a / d) for 0 <= a < 2^31 (Granlund-Montgomery; host computes mul/shr once per spec).
struct KsFastDiv {
  uint32_t mul, shr, d, pad;
};

// branch-free for every d >= 1: umulhi(2a, ceil(2^(31+l)/d)) >> l with l = ceil(log2 d); 2a fits because a < 2^31
KS_DEV uint32_t ks_div(uint32_t a, const KsFastDiv& f) { return __umulhi(a << 1, f.mul) >> f.shr; }
KS_DEV uint32_t ks_ceil_div(uint32_t a, const KsFastDiv& f) {
  uint32_t q = ks_div(a, f);
  return q + (q * f.d != a ? 1u : 0u);
}
// ceil(a / d) for 1 <= a < 2^31 as floor((a - 1) / d) + 1: four instructions instead of seven (a = 0 gives garbage:
// the caller selects 0 itself, usually together with a test it needs anyway)
KS_DEV uint32_t ks_ceil_div_pos(uint32_t a, const KsFastDiv& f) { return (__umulhi(2u * a - 2u, f.mul) >> f.shr) + 1u; }

// ------------------------------------------------------------------ per-spec constants (device form)
struct KsSpecDev {
  float inv_peak_flops, inv_peak_bw, t0, inv_t0;
  float l2_bytes, lg_ridge, inv_slots, slots_f;
  KsFastDiv tile_m, tile_n, ew, slots;
  float ar_alpha0, ar_inv_beta, pad0, pad1;       // Eq. 3
};
static_assert(sizeof(KsSpecDev) == 112, "KsSpecDev layout");

#define KS_MAX_SPECS_PER_LAUNCH 64

// per-bucket constants
struct KsBucketDev {
  const void* cols[KS_MAX_COLS];
  float* lat;          // [n_specs][n]
  int32_t* tiles;      // optional
  int32_t* waves;      // optional
  float* troof;        // optional
  int32_t family, n, col_f32, s;
  int32_t hq, hkv, hd, n_cols;
  // density routing (KS_TIER_B_ROUTED): when idx != nullptr the kernel works on the row LIST
  // idx[0 .. *count) instead of rows 0 .. n (outputs still go to the listed rows' own slots)
  const int32_t* idx;
  const int32_t* count;
};

// Tier-B grid constants
struct KsGridDev {
  const float* values;   // device, dims product floats
  int32_t dims[3];
  int32_t n_nodes;
  int32_t stride[3];     // element strides; 0 for a flat (1-node) axis
  int32_t pad;
  float lo[3];
  float scale[3];        // (dims-1)/(hi-lo); 0 for a flat axis
  int32_t vmin[3], vmax[3];   // the hull on integers: ceil(2^lo) <= v <= floor(2^hi) (INT_MIN/INT_MAX on a flat axis)
  int32_t* route_idx;    // KS_TIER_B_ROUTED pass 1: out-of-hull rows are appended here ...
  int32_t* route_count;  // ... at *route_count (zeroed before the launch); nullptr = plain Tier B
};

// ------------------------------------------------------------------ S1: descriptor decode
struct KsWork {
  float F, Y;       // F_comp [FLOP], F_mem [bytes]
  uint32_t B;       // CTA / tile count (saturates at INT32_MAX)
};

KS_DEV uint32_t ks_sat31(unsigned long long x) {
  const uint32_t hi = (uint32_t)(x >> 32), lo = (uint32_t)x;      // two 32-bit tests instead of a 64-bit compare
  return (hi != 0u || (int32_t)lo < 0) ? 0x7fffffffu : lo;
}
KS_DEV int ks_nonneg(int v) { return v > 0 ? v : 0; }

// elementwise sub-op tables (words moved / FLOPs per element), Q1
KS_DEV float ks_ew_rw(int op) { return (op == 1 || op == 5) ? 3.0f : 2.0f; }
KS_DEV float ks_ew_fl(int op) { return (float)((0x100644u >> (4 * op)) & 0xFu); }
KS_DEV int ks_ew_op(int op) { return op < 0 ? 0 : (op > 5 ? 5 : op); }

template <int FAM>
KS_DEV KsWork ks_decode(const int* v, const KsBucketDev& bk, const KsSpecDev& sp) {
  KsWork w;
  const float s = (float)bk.s;
  if (FAM == KS_FAM_GEMM) {
    const int M = ks_nonneg(v[0]), N = ks_nonneg(v[1]), K = ks_nonneg(v[2]);
    const float Mf = (float)M, Nf = (float)N, Kf = (float)K;
    w.F = 2.0f * Mf * Nf * Kf;
    w.Y = s * fmaf(Mf, Kf, fmaf(Kf, Nf, Mf * Nf));
    const uint32_t B = ks_sat31((unsigned long long)ks_ceil_div_pos(M, sp.tile_m) * ks_ceil_div_pos(N, sp.tile_n));
    w.B = (M == 0 || N == 0) ? 0u : B;
  } else if (FAM == KS_FAM_GROUPED_GEMM) {
    const int N = ks_nonneg(v[0]), K = ks_nonneg(v[1]);
    const uint32_t cn = ks_ceil_div(N, sp.tile_n);
    unsigned long long b = 0;
    float sum = 0.0f, act = 0.0f;
#pragma unroll
    for (int e = 0; e < KS_N_EXPERTS; ++e) {
      const int m = ks_nonneg(v[2 + e]);
      sum += (float)m;
      act += m > 0 ? 1.0f : 0.0f;
      b += (unsigned long long)ks_ceil_div(m, sp.tile_m) * cn;
    }
    const float Nf = (float)N, Kf = (float)K;
    w.F = 2.0f * Nf * Kf * sum;
    w.Y = s * fmaf(Kf, sum, fmaf(act * Kf, Nf, Nf * sum));
    w.B = ks_sat31(b);
  } else if (FAM == KS_FAM_ATTN) {
    const int Bq = ks_nonneg(v[0]), q = ks_nonneg(v[1]);
    int kv = ks_nonneg(v[2]);
    kv = kv < q ? q : kv;
    // causal pairs: cached history + own triangle: q (kv - q) + q (q + 1) / 2 in fp32
    // (every term is non-negative, so the three roundings stay at ~1e-7 relative; F needs 1e-5)
    const float qf = (float)q, Bf = (float)Bq, hd = (float)bk.hd;
    const float pairs = fmaf(qf, (float)(kv - q), 0.5f * qf * (qf + 1.0f));
    w.F = 4.0f * Bf * (float)bk.hq * hd * pairs;
    w.Y = s * 2.0f * Bf * hd * fmaf(qf, (float)bk.hq, (float)kv * (float)bk.hkv);
    const uint32_t B = ks_sat31((unsigned long long)Bq * (unsigned long long)bk.hq * ks_ceil_div_pos(q, sp.tile_m));
    w.B = q == 0 ? 0u : B;
  } else if (FAM == KS_FAM_ALLREDUCE) {
    w.F = 0.0f; w.Y = 0.0f; w.B = 0u;               // a communication row has no roofline (ks_allreduce)
  } else {
    const int n = ks_nonneg(v[0]);
    const int op = ks_ew_op(v[1]);
    w.Y = s * (float)n * ks_ew_rw(op);
    w.F = (float)n * ks_ew_fl(op);
    w.B = n == 0 ? 0u : ks_ceil_div_pos(n, sp.ew);
  }
  if (w.B == 0u) { w.F = 0.0f; w.Y = 0.0f; }
  return w;
}

// ------------------------------------------------------------------ TP all-reduce, Eq. 3
// t_ar = alpha0 + 2 (P - 1) / P * S / beta_eff; P <= 1 moves nothing
KS_DEV float ks_allreduce(const int* v, const KsSpecDev& sp) {
  const int S = ks_nonneg(v[0]), P = v[1];
  if (P <= 1) return sp.ar_alpha0;
  const float Pf = (float)P;
  return fmaf(__fdividef(2.0f * (Pf - 1.0f), Pf), (float)S * sp.ar_inv_beta, sp.ar_alpha0);
}

// ------------------------------------------------------------------ S2: roofline + wave quantization
struct KsRoof {
  uint32_t W;
  float u, t_comp, t_mem, t_roof;
};

KS_DEV KsRoof ks_roofline(const KsWork& w, const KsSpecDev& sp) {
  KsRoof r;
  if (w.B == 0u) { r.W = 0u; r.u = 1.0f; r.t_comp = 0.0f; r.t_mem = 0.0f; r.t_roof = 0.0f; return r; }
  r.W = ks_ceil_div_pos(w.B, sp.slots);             // B >= 1 here
  r.u = __fdividef((float)r.W * sp.slots_f, (float)w.B);
  r.t_comp = w.F * sp.inv_peak_flops;
  r.t_mem = w.Y * sp.inv_peak_bw;
  r.t_roof = fmaxf(r.t_comp * r.u, r.t_mem);
  return r;
}

// ------------------------------------------------------------------ accurate log2 of a positive integer-valued float
// log2(x) = exponent + lg2.approx(mantissa in [1,2)): the MUFU's absolute error bound (2^-22)
// applies on (0.5,2), so splitting keeps ~1e-7 absolute error at any magnitude.
KS_DEV float ks_log2_pos(float x) {
  const uint32_t b = __float_as_uint(x);
  const float e = (float)((int)(b >> 23) - 127);
  const float m = __uint_as_float((b & 0x007fffffu) | 0x3f800000u);
  return e + __log2f(m);
}

KS_DEV float ks_clip1(float x) { return fminf(fmaxf(x, -1.0f), 1.0f); }

// ------------------------------------------------------------------ S3: features (Q2)
// Writes x[0..NIN).  All continuous; zero row when B == 0.
template <int FAM, int NIN>
KS_DEV void ks_features(const int* v, const KsBucketDev& bk, const KsSpecDev& sp, const KsWork& w,
                        const KsRoof& r, float* x) {
#pragma unroll
  for (int i = 0; i < NIN; ++i) x[i] = 0.0f;
  if (w.B == 0u) return;
  const float lai = fmaxf(__log2f(w.F) - __log2f(w.Y), -10.0f);          // log2 max(AI, 2^-10)
  x[0] = ks_clip1(lai * 0.0625f);
  x[1] = ks_clip1((lai - sp.lg_ridge) * 0.0625f);
  x[2] = ks_clip1(__log2f((float)r.W) * 0.0625f);
  x[3] = __fdividef((float)w.B, (float)r.W * sp.slots_f);
  x[4] = ks_clip1(__log2f(fmaxf(r.t_roof * sp.inv_t0, 0.0009765625f)) * 0.0625f);
  x[5] = fminf(1.0f, __fdividef(sp.l2_bytes, w.Y));
  x[6] = ks_clip1(__log2f(fmaxf(__fdividef(r.t_comp * r.u, r.t_mem), 9.5367431640625e-07f)) * 0.05f);
  x[7] = ks_clip1(__log2f(fmaxf((float)w.B * sp.inv_slots, 0.0009765625f)) * 0.0625f);
  if (NIN <= 8) return;
  if (FAM == KS_FAM_GEMM) {
    x[8] = ks_clip1(__log2f(fmaxf((float)v[0], 1.0f)) * 0.0625f);
    x[9] = ks_clip1(__log2f(fmaxf((float)v[1], 1.0f)) * 0.0625f);
    x[10] = ks_clip1(__log2f(fmaxf((float)v[2], 1.0f)) * 0.0625f);
  } else if (FAM == KS_FAM_GROUPED_GEMM) {
    float sum = 0.0f;
#pragma unroll
    for (int e = 0; e < KS_N_EXPERTS; ++e) sum += (float)ks_nonneg(v[2 + e]);
    x[8] = ks_clip1(__log2f(fmaxf(sum, 1.0f)) * 0.0625f);
    x[9] = ks_clip1(__log2f(fmaxf((float)v[0], 1.0f)) * 0.0625f);
    x[10] = ks_clip1(__log2f(fmaxf((float)v[1], 1.0f)) * 0.0625f);
  } else if (FAM == KS_FAM_ATTN) {
    const int kv = v[2] < v[1] ? v[1] : v[2];
    x[8] = ks_clip1(__log2f(fmaxf((float)v[0], 1.0f)) * 0.0625f);
    x[9] = ks_clip1(__log2f(fmaxf((float)v[1], 1.0f)) * 0.0625f);
    x[10] = ks_clip1(__log2f(fmaxf((float)kv, 1.0f)) * 0.0625f);
  } else {
    const int op = ks_ew_op(v[1]);
    x[8] = ks_clip1(__log2f(fmaxf((float)v[0], 1.0f)) * 0.03125f);
    x[9] = ks_ew_rw(op) * 0.25f;
    x[10] = ks_ew_fl(op) * 0.125f;
  }
  x[11] = (float)bk.s * 0.25f;
  if (NIN <= 12) return;
  if (FAM == KS_FAM_GROUPED_GEMM) {
    float sum = 0.0f, mx = 0.0f, act = 0.0f;
#pragma unroll
    for (int e = 0; e < KS_N_EXPERTS; ++e) {
      const float m = (float)ks_nonneg(v[2 + e]);
      sum += m;
      mx = fmaxf(mx, m);
      act += m > 0.0f ? 1.0f : 0.0f;
    }
    const float inv = __frcp_rn(sum);
#pragma unroll
    for (int e = 0; e < KS_N_EXPERTS; ++e) x[12 + e] = (float)ks_nonneg(v[2 + e]) * inv;
    x[20] = mx * inv;                       // (max / mean) / 8 with 8 experts
    x[21] = act * 0.125f;
  }
}

// ------------------------------------------------------------------ column loads
KS_DEV int ks_load_col(const void* col, int i, bool f32) {
  return f32 ? __float2int_rn(__ldg((const float*)col + i)) : __ldg((const int*)col + i);
}
