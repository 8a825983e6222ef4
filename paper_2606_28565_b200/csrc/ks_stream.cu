// ks_stream.cu — the HBM-bound streaming kernels: descriptor decode + roofline + wave quantization
// (+ Tier-B trilinear interpolation from a shared-memory-resident grid) + launch floor.
// S1, S2, S4b, S5 of DESIGN.md §1.  PAPER.md:191 Eq. 2, :88 Fig. 2, :211 Tier B.
//
// Layout: SoA int32/fp32 columns; each thread owns 4 consecutive rows and moves them with 16-byte
// vector loads/stores (streaming cache hints: every byte is touched once).  Per-spec constants sit
// in the kernel-parameter constant bank.  Tier B stages the whole grid (<= 128 KiB) into shared
// memory once per persistent CTA (16-byte loads by all threads, overlapped with the first rows'
// column loads).  Tier B is issue-bound, not HBM-bound: ~170 instructions per query (three
// exponent+MUFU log2, clamp/floor/index per axis, eight shared-memory gathers, seven lerps) on
// top of the 62 of decode + roofline; ncu: issue slots 67 % busy with the 32 resident warps.
#include "ks_internal.h"
#include "ks_ptx.cuh"

namespace {

template <int FAM> struct NCols { static constexpr int v = 3; };
template <> struct NCols<KS_FAM_GROUPED_GEMM> { static constexpr int v = 10; };
template <> struct NCols<KS_FAM_ELEMWISE> { static constexpr int v = 2; };
template <> struct NCols<KS_FAM_ALLREDUCE> { static constexpr int v = 2; };

template <int NC, bool F32>
KS_DEV void load_rows4(const KsBucketDev& bk, int row0, int n, int (&v)[4][NC]) {
  if (row0 + 4 <= n) {
#pragma unroll
    for (int c = 0; c < NC; ++c) {
      if (F32) {
        const float4 f = __ldcs(reinterpret_cast<const float4*>(static_cast<const float*>(bk.cols[c]) + row0));
        v[0][c] = __float2int_rn(f.x); v[1][c] = __float2int_rn(f.y);
        v[2][c] = __float2int_rn(f.z); v[3][c] = __float2int_rn(f.w);
      } else {
        const int4 q = __ldcs(reinterpret_cast<const int4*>(static_cast<const int*>(bk.cols[c]) + row0));
        v[0][c] = q.x; v[1][c] = q.y; v[2][c] = q.z; v[3][c] = q.w;
      }
    }
  } else {
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int c = 0; c < NC; ++c) v[j][c] = (row0 + j < n) ? ks_load_col(bk.cols[c], row0 + j, F32) : 0;
  }
}

template <typename T>
KS_DEV void store4(T* base, long long off, int row0, int n, bool vec, T a, T b, T c, T d) {
  T* ptr = base + off + row0;
  if (vec && row0 + 4 <= n) {
    if (sizeof(T) == 4) {
      float4 q;
      q.x = *reinterpret_cast<float*>(&a); q.y = *reinterpret_cast<float*>(&b);
      q.z = *reinterpret_cast<float*>(&c); q.w = *reinterpret_cast<float*>(&d);
      __stcs(reinterpret_cast<float4*>(ptr), q);
    }
  } else {
    if (row0 + 0 < n) ptr[0] = a;
    if (row0 + 1 < n) ptr[1] = b;
    if (row0 + 2 < n) ptr[2] = c;
    if (row0 + 3 < n) ptr[3] = d;
  }
}

// Tier-B axis values (Q5): GEMM (M,N,K); GROUPED (sum m,N,K); ATTN (B,q,max(kv,q));
// ELEMWISE (n, 2^subop, 1) -> log2 coordinates.
template <int FAM>
KS_DEV void grid_log2_axes(const int* v, float (&lg)[3], bool (&pos)[3]) {
  float a[3];
  if (FAM == KS_FAM_GEMM) {
    a[0] = (float)v[0]; a[1] = (float)v[1]; a[2] = (float)v[2];
  } else if (FAM == KS_FAM_GROUPED_GEMM) {
    float sum = 0.0f;
#pragma unroll
    for (int e = 0; e < KS_N_EXPERTS; ++e) sum += (float)ks_nonneg(v[2 + e]);
    a[0] = sum; a[1] = (float)v[0]; a[2] = (float)v[1];
  } else if (FAM == KS_FAM_ATTN) {
    a[0] = (float)v[0]; a[1] = (float)v[1]; a[2] = (float)(v[2] < v[1] ? v[1] : v[2]);
  } else {
    a[0] = (float)v[0]; a[1] = 1.0f; a[2] = 1.0f;
  }
#pragma unroll
  for (int k = 0; k < 3; ++k) { pos[k] = a[k] > 0.0f; lg[k] = pos[k] ? ks_log2_pos(a[k]) : 0.0f; }
  if (FAM == KS_FAM_ELEMWISE) lg[1] = (float)ks_ew_op(v[1]);
}

// Density routing (Q16): inside the measured hull = inside the grid's box,
// decided on integers (ceil(2^lo) <= v <= floor(2^hi) per non-flat axis, bounds computed on the host).
template <int FAM>
KS_DEV bool in_hull(const int* v, const KsGridDev& g) {
  long long a[3];
  if (FAM == KS_FAM_GEMM) {
    a[0] = v[0]; a[1] = v[1]; a[2] = v[2];
  } else if (FAM == KS_FAM_GROUPED_GEMM) {
    long long sum = 0;
#pragma unroll
    for (int e = 0; e < KS_N_EXPERTS; ++e) sum += ks_nonneg(v[2 + e]);
    a[0] = sum; a[1] = v[0]; a[2] = v[1];
  } else if (FAM == KS_FAM_ATTN) {
    a[0] = v[0]; a[1] = v[1]; a[2] = v[2] < v[1] ? v[1] : v[2];
  } else {
    a[0] = v[0]; a[1] = 1; a[2] = 1;                 // (n, 2^subop, 1): axis 1 is checked on the sub-op below
  }
  bool in = true;
#pragma unroll
  for (int k = 0; k < 3; ++k) in = in && a[k] >= (long long)g.vmin[k] && a[k] <= (long long)g.vmax[k];
  if (FAM == KS_FAM_ELEMWISE) {
    const long long b = 1ll << ks_ew_op(v[1]);
    in = a[0] >= (long long)g.vmin[0] && a[0] <= (long long)g.vmax[0] && b >= (long long)g.vmin[1] && b <= (long long)g.vmax[1];
  }
  return in;
}

// trilinear interpolation of the stored efficiency; grid values in shared memory
template <int FAM>
KS_DEV float trilinear(const int* v, const KsGridDev& g, const float* __restrict__ sg) {
  float lg[3];
  bool pos[3];
  grid_log2_axes<FAM>(v, lg, pos);
  int base = 0;
  float f[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const float top = (float)(g.dims[a] - 1);
    float c = pos[a] ? (lg[a] - g.lo[a]) * g.scale[a] : 0.0f;
    c = fminf(fmaxf(c, 0.0f), top);                 // clamp to the measured span (fmaxf drops NaN)
    int i = (int)c;
    const int imax = g.dims[a] >= 2 ? g.dims[a] - 2 : 0;
    i = i > imax ? imax : i;
    f[a] = c - (float)i;
    base += i * g.stride[a];
  }
  const int s0 = g.stride[0], s1 = g.stride[1], s2 = g.stride[2];
  const float v000 = sg[base], v001 = sg[base + s2];
  const float v010 = sg[base + s1], v011 = sg[base + s1 + s2];
  const float v100 = sg[base + s0], v101 = sg[base + s0 + s2];
  const float v110 = sg[base + s0 + s1], v111 = sg[base + s0 + s1 + s2];
  const float c00 = fmaf(f[2], v001 - v000, v000), c01 = fmaf(f[2], v011 - v010, v010);
  const float c10 = fmaf(f[2], v101 - v100, v100), c11 = fmaf(f[2], v111 - v110, v110);
  const float c0 = fmaf(f[1], c01 - c00, c00), c1 = fmaf(f[1], c11 - c10, c10);
  return fmaf(f[0], c1 - c0, c0);
}

template <int FAM, int TIER, bool F32, bool ONE>
__global__ void __launch_bounds__(TIER == KS_TIER_B ? (FAM == KS_FAM_GROUPED_GEMM ? 512 : 1024) : 256)
ks_stream_kernel(const __grid_constant__ KsStreamParams p) {
  ks_launch_dependents();     // the next kernel of the stream may be scheduled now (it waits for us itself) ...
  cudaGridDependencySynchronize();   // ... as we wait for the one before us (ks_launch_pdl)
  constexpr int NC = NCols<FAM>::v;
  extern __shared__ __align__(128) float sgrid[];

  // row-list mode (the learned fallback of density routing): rows idx[0 .. *count) instead of 0 .. n
  const bool gather = TIER == KS_TIER_BOUNDED && p.bk.idx != nullptr;
  const int n = gather ? min(__ldg(p.bk.count), p.bk.n) : p.bk.n;
  const int n4 = (n + 3) >> 2;
  const int stride = gridDim.x * blockDim.x;
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  int v[4][NC];
  if (TIER == KS_TIER_B) {
    // first rows' columns are requested before the grid is staged, so the two overlap
    if (g < n4) load_rows4<NC, F32>(p.bk, g << 2, n, v);
    // stage the grid once per CTA with 16-byte loads by every thread (it is L2-resident after the
    // first CTA touched it; the values array is padded to a multiple of 4 floats)
    const int nv = (p.grid.n_nodes + 3) >> 2;
    const float4* __restrict__ src = reinterpret_cast<const float4*>(p.grid.values);
    float4* dst = reinterpret_cast<float4*>(sgrid);
    for (int i = threadIdx.x; i < nv; i += blockDim.x) dst[i] = __ldg(src + i);
    __syncthreads();
  }
  bool have = TIER == KS_TIER_B;                     // Tier B: the first trip's columns are already loaded
  for (; g < n4; g += stride) {
    const int row0 = g << 2;
    int rr[4] = {row0, row0 + 1, row0 + 2, row0 + 3};
    if (gather) {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        rr[j] = row0 + j < n ? __ldg(p.bk.idx + row0 + j) : 0;
#pragma unroll
        for (int c = 0; c < NC; ++c) v[j][c] = row0 + j < n ? ks_load_col(p.bk.cols[c], rr[j], F32) : 0;
      }
    } else if (!have) {
      load_rows4<NC, F32>(p.bk, row0, n, v);
    }
    have = false;
    if (TIER == KS_TIER_B && p.grid.route_idx != nullptr) {
      // density routing, pass 1: remember the rows outside the hull for the learned head (their
      // clamped Tier-B value written below is overwritten by pass 2, which runs after this kernel)
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (row0 + j < n && !in_hull<FAM>(v[j], p.grid)) p.grid.route_idx[atomicAdd(p.grid.route_count, 1)] = row0 + j;
    }

    float e[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) e[j] = 1.0f;
    if (TIER == KS_TIER_B) {
#pragma unroll
      for (int j = 0; j < 4; ++j) e[j] = fmaxf(trilinear<FAM>(v[j], p.grid, sgrid), 0.0009765625f);
    }

    // (Tier A, bounded analytical head: e depends on the spec through the features, see below)
    // ONE: a single spec -> its constants are read straight from the constant bank (no index math)
    const int n_specs = ONE ? 1 : p.n_specs;
    for (int s = 0; s < n_specs; ++s) {
      const KsSpecDev& sp = p.specs.s[ONE ? 0 : s];
      const long long off = (long long)s * p.spec_stride;
      const bool vec = ((off & 3ll) == 0);
      float t[4], tr[4];
      int tiles[4], waves[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const KsWork w = ks_decode<FAM>(v[j], p.bk, sp);
        const KsRoof r = ks_roofline(w, sp);
        tiles[j] = (int)w.B;
        waves[j] = (int)r.W;
        tr[j] = r.t_roof;
        // Eq. 2: t = max(t_roof * eta, t0), eta = 1/e; the floor is applied after eta
        if (TIER == KS_TIER_BOUNDED) {
          // bounded analytical head (Q15): e = gamma(x) - alpha(x) / W
          float x[KS_BOUNDED_NF];
          ks_features<FAM, KS_BOUNDED_NF>(v[j], p.bk, sp, w, r, x);
          float zg = p.bounded.b_gamma, za = p.bounded.b_alpha;
#pragma unroll
          for (int i = 0; i < KS_BOUNDED_NF; ++i) {
            zg = fmaf(p.bounded.w_gamma[i], x[i], zg);
            za = fmaf(p.bounded.w_alpha[i], x[i], za);
          }
          const float gamma = __fdividef(1.0f, 1.0f + __expf(-zg));
          const float ev = r.W > 0u ? gamma - __fdividef(fmaxf(za, 0.0f), (float)r.W) : gamma;
          e[j] = fmaxf(fminf(ev, 1.0f), 0.0009765625f);
        }
        t[j] = fmaxf(TIER == KS_TIER_NONE ? r.t_roof : __fdividef(r.t_roof, e[j]), sp.t0);
        if (FAM == KS_FAM_ALLREDUCE) tr[j] = t[j] = ks_allreduce(v[j], sp);   // Eq. 3 as it stands
      }
      if (gather) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if (row0 + j < n) {
            p.bk.lat[off + rr[j]] = t[j];
            if (p.bk.tiles) p.bk.tiles[off + rr[j]] = tiles[j];
            if (p.bk.waves) p.bk.waves[off + rr[j]] = waves[j];
            if (p.bk.troof) p.bk.troof[off + rr[j]] = tr[j];
          }
        }
        continue;
      }
      store4<float>(p.bk.lat, off, row0, n, vec, t[0], t[1], t[2], t[3]);
      if (p.bk.tiles) store4<int>(p.bk.tiles, off, row0, n, vec, tiles[0], tiles[1], tiles[2], tiles[3]);
      if (p.bk.waves) store4<int>(p.bk.waves, off, row0, n, vec, waves[0], waves[1], waves[2], waves[3]);
      if (p.bk.troof) store4<float>(p.bk.troof, off, row0, n, vec, tr[0], tr[1], tr[2], tr[3]);
    }
  }
}

template <int FAM, int TIER>
cudaError_t launch_ft(const KsStreamParams& p, int num_sms, cudaStream_t st) {
  const int n4 = (p.bk.n + 3) >> 2;
  if (n4 == 0) return cudaSuccess;
  const bool f32 = p.bk.col_f32 != 0;
  if (TIER == KS_TIER_B) {
    const int threads = FAM == KS_FAM_GROUPED_GEMM ? 512 : 1024;   // 10 columns x 4 rows need > 64 registers
    const size_t smem = (size_t)((p.grid.n_nodes + 3) & ~3) * 4;
    int blocks = (n4 + threads - 1) / threads;
    if (blocks > num_sms) blocks = num_sms;          // persistent: one CTA per SM, grid staged once
    const bool one = p.n_specs == 1;
    auto kern = f32 ? (one ? ks_stream_kernel<FAM, TIER, true, true> : ks_stream_kernel<FAM, TIER, true, false>)
                    : (one ? ks_stream_kernel<FAM, TIER, false, true> : ks_stream_kernel<FAM, TIER, false, false>);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    return ks_launch_pdl(kern, blocks, threads, smem, st, p);
  } else {
    const int threads = 256;
    int blocks = (n4 + threads - 1) / threads;
    const int cap = num_sms * 8 * 4;                 // up to 4 waves of 8 resident CTAs per SM
    if (blocks > cap) blocks = cap - (cap % num_sms);
    const bool one = p.n_specs == 1;
    auto kern = f32 ? (one ? ks_stream_kernel<FAM, TIER, true, true> : ks_stream_kernel<FAM, TIER, true, false>)
                    : (one ? ks_stream_kernel<FAM, TIER, false, true> : ks_stream_kernel<FAM, TIER, false, false>);
    // launched programmatically dependent (ks_launch_pdl): measured on cfg4a, back to back: GEMM 37.0 -> 35.3 us,
    // attention 16.5 -> 13.9 us, elementwise 31.1 -> 29.1 us
    return ks_launch_pdl(kern, blocks, threads, 0, st, p);
  }
  return cudaGetLastError();
}

template <int TIER>
cudaError_t launch_t(const KsStreamParams& p, int num_sms, cudaStream_t st) {
  switch (p.bk.family) {
    case KS_FAM_GEMM: return launch_ft<KS_FAM_GEMM, TIER>(p, num_sms, st);
    case KS_FAM_GROUPED_GEMM: return launch_ft<KS_FAM_GROUPED_GEMM, TIER>(p, num_sms, st);
    case KS_FAM_ATTN: return launch_ft<KS_FAM_ATTN, TIER>(p, num_sms, st);
    case KS_FAM_ELEMWISE: return launch_ft<KS_FAM_ELEMWISE, TIER>(p, num_sms, st);
    case KS_FAM_ALLREDUCE: return launch_ft<KS_FAM_ALLREDUCE, KS_TIER_NONE>(p, num_sms, st);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace

namespace {

template <int FAM, int NC>
KS_DEV void small_row(const KsStreamSmallParams& p, const KsBucketDev& bk, const int i) {
  int v[NC];
#pragma unroll
  for (int c = 0; c < NC; ++c)
    v[c] = bk.col_f32 ? __float2int_rn(__ldg(static_cast<const float*>(bk.cols[c]) + i))
                      : __ldg(static_cast<const int*>(bk.cols[c]) + i);
  for (int s = 0; s < p.n_specs; ++s) {
    const KsSpecDev& sp = p.specs.s[s];
    const KsWork w = ks_decode<FAM>(v, bk, sp);
    const KsRoof r = ks_roofline(w, sp);
    float tr = r.t_roof, t = fmaxf(r.t_roof, sp.t0);            // Eq. 2 with eta = 1: floor after eta
    if (FAM == KS_FAM_ALLREDUCE) tr = t = ks_allreduce(v, sp);  // Eq. 3 as it stands
    const long long o = (long long)s * bk.n + i;
    bk.lat[o] = t;
    if (bk.tiles) bk.tiles[o] = (int)w.B;
    if (bk.waves) bk.waves[o] = (int)r.W;
    if (bk.troof) bk.troof[o] = tr;
  }
}

__global__ void __launch_bounds__(256) ks_stream_small_kernel(const __grid_constant__ KsStreamSmallParams p) {
  ks_launch_dependents();
  cudaGridDependencySynchronize();
  const int g = blockIdx.x * 256 + threadIdx.x;
  if (g >= p.row_begin[p.n_buckets]) return;
  int b = 0;
  while (g >= p.row_begin[b + 1]) ++b;
  const KsBucketDev& bk = p.bk[b];
  const int i = g - p.row_begin[b];
  switch (bk.family) {
    case KS_FAM_GEMM: small_row<KS_FAM_GEMM, 3>(p, bk, i); break;
    case KS_FAM_GROUPED_GEMM: small_row<KS_FAM_GROUPED_GEMM, 10>(p, bk, i); break;
    case KS_FAM_ATTN: small_row<KS_FAM_ATTN, 3>(p, bk, i); break;
    case KS_FAM_ELEMWISE: small_row<KS_FAM_ELEMWISE, 2>(p, bk, i); break;
    default: small_row<KS_FAM_ALLREDUCE, 2>(p, bk, i); break;
  }
}

}  // namespace

cudaError_t ks_launch_stream_small(const KsStreamSmallParams& p, cudaStream_t st) {
  const int n = p.row_begin[p.n_buckets];
  if (n <= 0) return cudaSuccess;
  return ks_launch_pdl(ks_stream_small_kernel, (n + 255) / 256, 256, 0, st, p);
}

cudaError_t ks_launch_stream(const KsStreamParams& p, int num_sms, cudaStream_t st) {
  if (p.tier == KS_TIER_BOUNDED) return launch_t<KS_TIER_BOUNDED>(p, num_sms, st);
  return p.tier == KS_TIER_B ? launch_t<KS_TIER_B>(p, num_sms, st) : launch_t<KS_TIER_NONE>(p, num_sms, st);
}
