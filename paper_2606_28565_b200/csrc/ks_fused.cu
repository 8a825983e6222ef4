// ks_fused.cu — one pass of the whole Tier-NONE hot path in ONE kernel: S1 descriptor decode, S2 roofline + wave
// quantization, S5 launch floor (PAPER.md:191 Eq. 2, :88 Fig. 2), S6 step sums and S7 Eq. 4
// (PAPER.md:233), for ks_run_steps(KS_MEM_DEVICE, KS_TIER_NONE) with one spec vector (config 4a: 100,000 serving
// steps, 29.9M kernel instances; with per-row multiplicities also the pass ks_sim_run makes every iteration).
//
// ks_predict_kernels + ks_compose_steps write every per-kernel latency to HBM and read it back (2 x 120 MB of the
// 548 MB a config-4a step moves).  Here the step kernel's staging phase COMPUTES the latencies instead of copying
// them: one CTA per chunk of 32 consecutive steps (rows of a bucket are step-sorted, so the chunk is one contiguous
// row range of every bucket), every thread takes aligned groups of 4 consecutive rows (16-byte column loads, the
// streaming kernel's arithmetic: same device functions, same bits), writes the four latencies into the chunk's
// shared-memory image — laid out exactly as ks_compose_kernel lays out its staged copy — and, when the caller wants
// the per-kernel latencies, to HBM as well; then the same eight-lanes-per-step reduction and Eq. 4 epilogue as
// ks_compose_kernel.  The step latencies are therefore bit-identical to the two-call path's (staged chunks), the
// per-kernel latencies too, and without a latency output a step moves the descriptor columns only (307 MB).
// A chunk that does not fit the staging buffer is summed by a warp per step straight from the columns.
// No atomics: bit-reproducible.
#include "ks_internal.h"
#include "ks_ptx.cuh"

namespace {

constexpr int kWarps = 16;             // 512 threads, four CTAs per SM: 2,048 threads per SM like the streaming kernel
constexpr int kThreads = kWarps * 32;
constexpr int kS = 32;                 // steps per chunk = ks_compose.cu's kS (same shared-memory image)
constexpr int kCapFloats = 12032;      // = ks_compose.cu's kCapFloats: 47 KiB, four CTAs per SM
constexpr int kSlackFloats = 192;

template <int FAM> struct NCols { static constexpr int v = 3; };
template <> struct NCols<KS_FAM_ELEMWISE> { static constexpr int v = 2; };
template <> struct NCols<KS_FAM_ALLREDUCE> { static constexpr int v = 2; };

// Eq. 2 with eta = 1 (Tier NONE): t = max(t_roof, t0); an all-reduce row is Eq. 3 as it stands
template <int FAM>
KS_DEV float row_latency(const int* v, const KsBucketDev& bk, const KsSpecDev& sp) {
  if (FAM == KS_FAM_ALLREDUCE) return ks_allreduce(v, sp);
  const KsWork w = ks_decode<FAM>(v, bk, sp);
  const KsRoof r = ks_roofline(w, sp);
  return fmaxf(r.t_roof, sp.t0);
}

template <int NC>
KS_DEV void load_rows4(const KsBucketDev& bk, int row0, int (&v)[4][NC]) {
  if (row0 + 4 <= bk.n) {
#pragma unroll
    for (int c = 0; c < NC; ++c) {
      const int4 q = __ldcs(reinterpret_cast<const int4*>(static_cast<const int*>(bk.cols[c]) + row0));
      v[0][c] = q.x; v[1][c] = q.y; v[2][c] = q.z; v[3][c] = q.w;
    }
  } else {
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int c = 0; c < NC; ++c) v[j][c] = row0 + j < bk.n ? __ldg(static_cast<const int*>(bk.cols[c]) + row0 + j) : 0;
  }
}

// latencies of rows [a0, a0 + len) of one bucket (a0, len multiples of 4) -> dst[0, len); rows inside the chunk
// [lo, hi) also go to bk.lat when the caller wants them (a group on the chunk's edge is shared with the
// neighbouring chunk: each CTA writes only its own rows).  MULT (layer-homogeneous form): a row stands
// for m_k identical kernels; the image holds m_k t_k and a second image dstm the multiplicities (Eq. 4's n = sum m_k)
template <int FAM, bool MULT>
KS_DEV void stage_bucket(const KsBucketDev& bk, const int32_t* __restrict__ mult, const KsSpecDev& sp, const int a0, const int len,
                         const int lo, const int hi, float* __restrict__ dst, int* __restrict__ dstm, const int tid) {
  constexpr int NC = NCols<FAM>::v;
#pragma unroll 1
  for (int i = tid * 4; i < len; i += kThreads * 4) {
    const int row0 = a0 + i;
    int v[4][NC];
    load_rows4<NC>(bk, row0, v);
    int4 m = make_int4(1, 1, 1, 1);
    if (MULT && mult != nullptr) {
      if (row0 + 4 <= bk.n) {
        m = __ldg(reinterpret_cast<const int4*>(mult + row0));
      } else {
        m.x = row0 + 0 < bk.n ? __ldg(mult + row0 + 0) : 0; m.y = row0 + 1 < bk.n ? __ldg(mult + row0 + 1) : 0;
        m.z = row0 + 2 < bk.n ? __ldg(mult + row0 + 2) : 0; m.w = row0 + 3 < bk.n ? __ldg(mult + row0 + 3) : 0;
      }
    }
    float4 t;
    t.x = row_latency<FAM>(v[0], bk, sp); t.y = row_latency<FAM>(v[1], bk, sp);
    t.z = row_latency<FAM>(v[2], bk, sp); t.w = row_latency<FAM>(v[3], bk, sp);
    if (bk.lat) {
      if (row0 >= lo && row0 + 4 <= hi) {
        __stcs(reinterpret_cast<float4*>(bk.lat + row0), t);
      } else {
        if (row0 + 0 >= lo && row0 + 0 < hi) bk.lat[row0 + 0] = t.x;
        if (row0 + 1 >= lo && row0 + 1 < hi) bk.lat[row0 + 1] = t.y;
        if (row0 + 2 >= lo && row0 + 2 < hi) bk.lat[row0 + 2] = t.z;
        if (row0 + 3 >= lo && row0 + 3 < hi) bk.lat[row0 + 3] = t.w;
      }
    }
    if (MULT) {
      t.x *= (float)m.x; t.y *= (float)m.y; t.z *= (float)m.z; t.w *= (float)m.w;
      *reinterpret_cast<int4*>(dstm + i) = m;
    }
    *reinterpret_cast<float4*>(dst + i) = t;
  }
}

// this lane's share (rows beg + lane, beg + lane + 32, ...) of one step of one bucket, straight from the columns
template <int FAM, bool MULT>
KS_DEV float lane_rows(const KsBucketDev& bk, const int32_t* __restrict__ mult, const KsSpecDev& sp, const int beg, const int end,
                       const int lane, int& cnt) {
  constexpr int NC = NCols<FAM>::v;
  float acc = 0.0f;
#pragma unroll 1
  for (int r = beg + lane; r < end; r += 32) {
    int v[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) v[c] = __ldg(static_cast<const int*>(bk.cols[c]) + r);
    const float t = row_latency<FAM>(v, bk, sp);
    if (bk.lat) bk.lat[r] = t;
    const int m = (MULT && mult != nullptr) ? __ldg(mult + r) : 1;
    acc += MULT ? t * (float)m : t;
    cnt += m;
  }
  return acc;
}

// NB = bound on the bucket count (1-4: exact, or 8); MULT: some bucket carries multiplicities
template <int NB, bool MULT>
__global__ void __launch_bounds__(kThreads, 4)   // <= 32 registers
ks_fused_none_kernel(const __grid_constant__ KsFusedParams p) {
  extern __shared__ __align__(128) float sdata[];
  __shared__ int offs[NB][kS + 1];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int s0 = (int)blockIdx.x * kS;
  const int ns = p.n_steps - s0 < kS ? p.n_steps - s0 : kS;

  ks_launch_dependents();            // the totals kernel may be scheduled under this one ...
  cudaGridDependencySynchronize();   // ... as this one waits for whatever precedes it on the stream (ks_launch_pdl)
  for (int idx = tid; idx < NB * (kS + 1); idx += kThreads) {
    const int b = idx / (kS + 1), j = idx - b * (kS + 1);
    offs[b][j] = b < p.n_batches ? __ldg(p.step_off[b] + (s0 + j < p.n_steps ? s0 + j : p.n_steps)) : 0;
  }
  __syncthreads();

  // the chunk's shared-memory image: per bucket the rows [a0, a1) (aligned out to groups of 4), back to back
  int sbase[NB];
  int used = 0;
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    const int a0 = offs[b][0] & ~3;
    sbase[b] = used - a0;
    used += ((offs[b][kS] + 3) & ~3) - a0;
  }
  const KsSpecDev& sp = p.spec;
  // MULT: the multiplicities' image (ints) sits behind the latencies' in the same buffer
  const int cap = MULT ? (p.cap_floats >> 1) & ~3 : p.cap_floats;
  int* smul = reinterpret_cast<int*>(sdata) + cap;
  if (used <= cap) {
    // (sharing the groups out over the threads across all buckets -- five full trips per config-4a chunk instead of
    // 3 + 1 + 3 partly empty ones -- was measured: 6 % slower; the kernel is bound by issue slots, not by trips)
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      if (b >= p.n_batches) break;
      const KsBucketDev& bk = p.bk[b];
      const int32_t* mu = p.mult[b];
      const int lo = offs[b][0], hi = offs[b][kS], a0 = lo & ~3, len = ((hi + 3) & ~3) - a0;
      float* dst = sdata + (sbase[b] + a0);
      int* dstm = smul + (sbase[b] + a0);
      switch (bk.family) {                                            // CTA-uniform
        case KS_FAM_GEMM: stage_bucket<KS_FAM_GEMM, MULT>(bk, mu, sp, a0, len, lo, hi, dst, dstm, tid); break;
        case KS_FAM_ATTN: stage_bucket<KS_FAM_ATTN, MULT>(bk, mu, sp, a0, len, lo, hi, dst, dstm, tid); break;
        case KS_FAM_ELEMWISE: stage_bucket<KS_FAM_ELEMWISE, MULT>(bk, mu, sp, a0, len, lo, hi, dst, dstm, tid); break;
        default: stage_bucket<KS_FAM_ALLREDUCE, MULT>(bk, mu, sp, a0, len, lo, hi, dst, dstm, tid); break;
      }
    }
    __syncthreads();
    // EIGHT LANES PER STEP over aligned 16-byte groups: ks_compose_kernel's reduce_wide, statement for statement (the
    // summation order, hence the bits, are those of the two-call path)
    const int sub = lane >> 3, l8 = lane & 7;
    const float4* __restrict__ s4 = reinterpret_cast<const float4*>(sdata);
    const int4* __restrict__ m4 = reinterpret_cast<const int4*>(smul);
#pragma unroll 1
    for (int j = warp * 4 + sub; j < kS; j += kWarps * 4) {
      const bool valid = j < ns;
      float acc = 0.0f;
      int cnt = 0;
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        const int beg = valid ? offs[b][j] : 0, end = valid ? offs[b][j + 1] : 0;
        const int P = sbase[b] + beg, Q = sbase[b] + end;
        if (!MULT && l8 == 0) cnt += end - beg;
        if (Q > P) {
          const int G0 = P >> 2, G1 = (Q + 3) >> 2;
          float a0s = 0.0f, a1s = 0.0f, a2s = 0.0f, a3s = 0.0f;
#pragma unroll 1
          for (int g = G0 + 1 + l8; g < G1 - 1; g += 8) {
            const float4 v = s4[g];
            ks_add2(a0s, a1s, a0s, a1s, v.x, v.y);
            ks_add2(a2s, a3s, a2s, a3s, v.z, v.w);
            if (MULT) { const int4 m = m4[g]; cnt += (m.x + m.y) + (m.z + m.w); }
          }
          if (l8 == 0 || (l8 == 1 && G1 - 1 > G0)) {
            const int g = l8 == 0 ? G0 : G1 - 1, e0 = 4 * g;
            const float4 v = s4[g];
            a0s += (e0 >= P && e0 < Q) ? v.x : 0.0f;
            a1s += (e0 + 1 >= P && e0 + 1 < Q) ? v.y : 0.0f;
            a2s += (e0 + 2 >= P && e0 + 2 < Q) ? v.z : 0.0f;
            a3s += (e0 + 3 >= P && e0 + 3 < Q) ? v.w : 0.0f;
            if (MULT) {
              const int4 m = m4[g];
              cnt += ((e0 >= P && e0 < Q) ? m.x : 0) + ((e0 + 1 >= P && e0 + 1 < Q) ? m.y : 0) +
                     ((e0 + 2 >= P && e0 + 2 < Q) ? m.z : 0) + ((e0 + 3 >= P && e0 + 3 < Q) ? m.w : 0);
            }
          }
          acc += (a0s + a1s) + (a2s + a3s);
        }
      }
      acc += __shfl_xor_sync(0xffffffffu, acc, 4);
      acc += __shfl_xor_sync(0xffffffffu, acc, 2);
      acc += __shfl_xor_sync(0xffffffffu, acc, 1);
      if (MULT) {                                                     // per-lane partial launch counts (exact: integers)
        cnt += __shfl_xor_sync(0xffffffffu, cnt, 4);
        cnt += __shfl_xor_sync(0xffffffffu, cnt, 2);
        cnt += __shfl_xor_sync(0xffffffffu, cnt, 1);
      }
      if (l8 == 0 && valid) {
        const float t_gpu = p.sp.body_scale * acc;
        // Eq. 4: t_step = max(t_gpu + n c_disp, l) + max(0, c_ovl - t_gpu) + c_tail
        const float t = fmaxf(fmaf((float)cnt, p.sp.c_disp, t_gpu), p.sp.floor_l) +
                        fmaxf(0.0f, p.sp.c_ovl - t_gpu) + p.sp.c_tail;
        p.step_lat[s0 + j] = t;
      }
    }
  } else {
    // very long steps: a warp per step, lanes stride the step's rows of every bucket, fixed-order shuffle tree
#pragma unroll 1
    for (int j = warp; j < ns; j += kWarps) {
      float acc = 0.0f;
      int cnt = 0;
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        if (b >= p.n_batches) break;
        const KsBucketDev& bk = p.bk[b];
        const int32_t* mu = p.mult[b];
        const int beg = offs[b][j], end = offs[b][j + 1];
        switch (bk.family) {
          case KS_FAM_GEMM: acc += lane_rows<KS_FAM_GEMM, MULT>(bk, mu, sp, beg, end, lane, cnt); break;
          case KS_FAM_ATTN: acc += lane_rows<KS_FAM_ATTN, MULT>(bk, mu, sp, beg, end, lane, cnt); break;
          case KS_FAM_ELEMWISE: acc += lane_rows<KS_FAM_ELEMWISE, MULT>(bk, mu, sp, beg, end, lane, cnt); break;
          default: acc += lane_rows<KS_FAM_ALLREDUCE, MULT>(bk, mu, sp, beg, end, lane, cnt); break;
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        acc += __shfl_xor_sync(0xffffffffu, acc, o);
        cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
      }
      if (lane == 0) {
        const float t_gpu = p.sp.body_scale * acc;
        const float t = fmaxf(fmaf((float)cnt, p.sp.c_disp, t_gpu), p.sp.floor_l) +
                        fmaxf(0.0f, p.sp.c_ovl - t_gpu) + p.sp.c_tail;
        p.step_lat[s0 + j] = t;
      }
    }
  }
}

}  // namespace

bool ks_fused_none_supported(int family, bool col_f32) {
  return !col_f32 && (family == KS_FAM_GEMM || family == KS_FAM_ATTN || family == KS_FAM_ELEMWISE || family == KS_FAM_ALLREDUCE);
}

cudaError_t ks_launch_fused_none(const KsFusedParams& p, cudaStream_t st) {
  if (p.n_steps <= 0 || p.n_batches < 1 || p.n_batches > KS_FUSED_MAX_BUCKETS) return cudaErrorInvalidValue;
  bool weighted = false;
  for (int b = 0; b < p.n_batches; ++b) weighted = weighted || p.mult[b] != nullptr;
  void (*kern)(const KsFusedParams);
  if (weighted)
    kern = p.n_batches <= 4 ? ks_fused_none_kernel<4, true> : ks_fused_none_kernel<8, true>;
  else
    kern = p.n_batches == 1 ? ks_fused_none_kernel<1, false> : p.n_batches == 2 ? ks_fused_none_kernel<2, false> :
           p.n_batches == 3 ? ks_fused_none_kernel<3, false> : p.n_batches == 4 ? ks_fused_none_kernel<4, false> :
                                                                                  ks_fused_none_kernel<8, false>;
  KsFusedParams q = p;
  q.cap_floats = kCapFloats;
  const size_t smem = (size_t)(kCapFloats + kSlackFloats) * 4;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  return ks_launch_pdl(kern, (unsigned)((p.n_steps + kS - 1) / kS), kThreads, smem, st, q);
}

int ks_fused_none_cap_floats(bool weighted) { return weighted ? kCapFloats / 2 : kCapFloats; }
