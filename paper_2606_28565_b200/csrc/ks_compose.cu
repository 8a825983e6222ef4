// ks_compose.cu — S6/S7: segmented reduction of kernel latencies into per-step GPU bodies
// (PAPER.md:231), the host-overlap step formula (Eq. 4) and per-configuration totals.
//
// ks_compose_kernel: one CTA per chunk of 32 consecutive steps (rows of a bucket are step-sorted, so
// a chunk is one contiguous range of every bucket's latency array).  The CTA reads the chunk's CSR
// bounds, then stages every bucket's range into shared memory with 16-byte cp.async copies (fire
// and forget: ~38 KB in flight per CTA, four CTAs per SM, no registers tied up), and its eight warps
// sum two steps at a time out of shared memory: per bucket the lanes read consecutive elements
// (conflict-free LDS with immediate offsets), ten loads per step pair issued before the first add,
// masked afterwards; one fixed-order shuffle tree per step; Eq. 4 epilogue.  No atomics:
// bit-reproducible.  A chunk that does not fit the buffer (very long steps) is summed straight
// from global memory by the same loop.
// Measured alternatives (profiles/README.md): persistent CTAs with 1-D TMA bulk copies (2-4 stages,
// with and without a producer warp), persistent cp.async double buffering, and persistent warps
// reading global memory directly were all slower (34-60 us against 31 us on cfg4a).
// Config totals: one CTA per (spec, config), fp64 accumulation.
#include "ks_internal.h"
#include "ks_ptx.cuh"

#include <type_traits>

namespace {

constexpr int kWarps = 8;
constexpr int kThreads = kWarps * 32;

constexpr int kS = 32;                 // steps per chunk (one CTA); small problems use kSmallS (more, lighter CTAs)
constexpr int kSmallS = 8;
constexpr int kSmallSteps = 16384;     // n_steps x n_specs up to which the small chunk is used
constexpr int kCapFloats = 12032;      // staged floats per CTA (47 KiB + slack): four CTAs per SM
constexpr int kCapFloatsBig = 18432;   // ... for workloads whose average chunk does not fit that: 72 KiB, three CTAs per SM
constexpr int kSlackFloats = 192;      // readable floats behind the staged data (masked lanes of the last step)

KS_DEV int mA_n(int n, int lane) { return n - lane; }   // elements 32 r < n - lane belong to this lane

// this lane's share of src[0, n) beyond the first 160 elements (rare: very long steps)
KS_DEV float lane_tail(const float* __restrict__ src, int n, int lane) {
  float a0 = 0.0f, a1 = 0.0f;
  int k = lane + 160;
#pragma unroll 1
  for (; k + 32 < n; k += 64) { a0 += src[k]; a1 += src[k + 32]; }
  if (k < n) a0 += src[k];
  return a0 + a1;
}

// NB = compile-time bound on the bucket count (1-4: exact, or 8)
template <int NB, bool MULT, int KS>
__global__ void __launch_bounds__(kThreads, 4)
ks_compose_kernel(const __grid_constant__ KsComposeParams p) {
  extern __shared__ __align__(128) float sdata[];
  __shared__ int offs[NB][KS + 1];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned cps = (unsigned)(p.n_steps + KS - 1) / KS;        // chunks per spec
  const unsigned spec = blockIdx.x / cps;
  const int s0 = (int)(blockIdx.x - spec * cps) * KS;
  const int ns = p.n_steps - s0 < KS ? p.n_steps - s0 : KS;

  // launched with programmatic stream serialization: the launch itself overlaps the tail of the
  // prediction kernel; nothing it produced (nor anything copied in for this call) is read before this
  ks_launch_dependents();            // ... and the totals kernel may be scheduled under this one
  cudaGridDependencySynchronize();
  for (int idx = tid; idx < p.n_batches * (KS + 1); idx += kThreads) {
    const int b = idx / (KS + 1), j = idx - b * (KS + 1);
    offs[b][j] = __ldg(p.step_off[b] + (s0 + j < p.n_steps ? s0 + j : p.n_steps));
  }
  __syncthreads();

  // The chunk's kernels are one contiguous range per bucket: stage all of them with 16-byte
  // cp.async copies (fire and forget: ~38 KB in flight per CTA, four CTAs per SM).
  int sbase[NB], len[NB];
  long long a0[NB];
  int used = 0;
  bool staged = true;
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    sbase[b] = 0; len[b] = 0; a0[b] = 0;
    if (b < p.n_batches) {
      const long long sb = (long long)spec * p.spec_stride[b];
      a0[b] = (sb + offs[b][0]) & ~3ll;
      long long a1 = (sb + offs[b][KS] + 3) & ~3ll;
      const long long tot = ((long long)p.n_specs * p.spec_stride[b]) & ~3ll;
      if (a1 > tot) a1 = tot;                                     // never read past the array end ...
      if (a1 < sb + offs[b][KS]) staged = false;                  // ... (its last < 4 floats: global path)
      len[b] = (int)(a1 - a0[b]);
      sbase[b] = used + (int)(sb - a0[b]);
      used += len[b];
    }
  }
  if (used > p.cap_floats) staged = false;                        // very long steps: straight from global
  // Multiplicities (shared by all specs) ride in the same cp.async group behind the latencies when they fit:
  // a chunk then costs one trip to memory for all buckets instead of one per bucket inside the reduction —
  // which matters when the arrays live in pinned host memory (the simulation loop reads its arena in place).
  int mbase[NB], mlen[NB], m0[NB];
  bool mstaged = MULT && staged;
  int* smult = reinterpret_cast<int*>(sdata + ((used + 3) & ~3));
  int mused = 0;
  if (MULT) {
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      mbase[b] = 0; mlen[b] = 0; m0[b] = 0;
      if (b < p.n_batches && p.mult[b] != nullptr) {
        m0[b] = offs[b][0] & ~3;
        int m1 = (offs[b][KS] + 3) & ~3;
        const int tot = (int)(p.spec_stride[b] & ~3ll);
        if (m1 > tot) m1 = tot;
        if (m1 < offs[b][KS] || (reinterpret_cast<uintptr_t>(p.mult[b]) & 15u) != 0) mstaged = false;
        mlen[b] = m1 - m0[b];
        mbase[b] = mused - m0[b];
        mused += mlen[b];
      }
    }
    if (((used + 3) & ~3) + mused > p.cap_floats) mstaged = false;
  }
  if (staged) {
    int base = 0;
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      if (b < p.n_batches) {
        const float* __restrict__ src = p.lat[b] + a0[b];
        for (int i = tid * 4; i < len[b]; i += kThreads * 4) ks_cp_async16(sdata + base + i, src + i);
        base += len[b];
      }
    }
    if (MULT && mstaged) {
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        if (b < p.n_batches && p.mult[b] != nullptr) {
          const int32_t* __restrict__ src = p.mult[b] + m0[b];
          int* dst = smult + mbase[b] + m0[b];
          for (int i = tid * 4; i < mlen[b]; i += kThreads * 4) ks_cp_async16(dst + i, src + i);
        }
      }
    }
    ks_cp_async_commit();
    ks_cp_async_wait<0>();
    __syncthreads();
  }

  // a warp sums two steps at a time (w and w + 8, then w + 16 and w + 24): per bucket ten independent
  // predicated loads before the first add, one fixed-order shuffle tree per step.  Two copies of
  // the loop so that the staged one uses 32-bit shared-memory addressing (LDS), not generic loads.
  auto reduce_all = [&](auto staged_tag) {
    constexpr bool STAGED = decltype(staged_tag)::value;
#pragma unroll 1
    for (int jA = warp; jA < ns; jA += 2 * kWarps) {
      const int jB = jA + kWarps;
      const bool hasB = jB < ns;
      float accA = 0.0f, accB = 0.0f;
      int cntA = 0, cntB = 0;
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        if (b < p.n_batches) {
          const int begA = offs[b][jA], nA = offs[b][jA + 1] - begA;
          const int begB = hasB ? offs[b][jB] : begA, nB = hasB ? offs[b][jB + 1] - begB : 0;
          const float* __restrict__ sA;
          const float* __restrict__ sB;
          if (STAGED) {
            sA = sdata + (sbase[b] + begA + lane);
            sB = sdata + (sbase[b] + begB + lane);
          } else {
            const float* base = p.lat[b] + (long long)spec * p.spec_stride[b];
            sA = base + begA + lane;
            sB = base + begB + lane;
          }
          const int mA = nA - lane, mB = nB - lane;                // this lane owns elements 32 r < m
          float x0, x1, x2, x3, x4, y0, y1, y2, y3, y4;
          if (STAGED) {
            // unconditional LDS with immediate offsets (the buffer has 160 floats of slack behind the
            // staged data, so every address is valid), masked after all ten loads are issued
            x0 = sA[0]; x1 = sA[32]; x2 = sA[64]; x3 = sA[96]; x4 = sA[128];
            y0 = sB[0]; y1 = sB[32]; y2 = sB[64]; y3 = sB[96]; y4 = sB[128];
            x0 = 0 < mA ? x0 : 0.0f; x1 = 32 < mA ? x1 : 0.0f; x2 = 64 < mA ? x2 : 0.0f;
            x3 = 96 < mA ? x3 : 0.0f; x4 = 128 < mA ? x4 : 0.0f;
            y0 = 0 < mB ? y0 : 0.0f; y1 = 32 < mB ? y1 : 0.0f; y2 = 64 < mB ? y2 : 0.0f;
            y3 = 96 < mB ? y3 : 0.0f; y4 = 128 < mB ? y4 : 0.0f;
          } else {
            x0 = 0 < mA ? sA[0] : 0.0f; y0 = 0 < mB ? sB[0] : 0.0f;
            x1 = 32 < mA ? sA[32] : 0.0f; y1 = 32 < mB ? sB[32] : 0.0f;
            x2 = 64 < mA ? sA[64] : 0.0f; y2 = 64 < mB ? sB[64] : 0.0f;
            x3 = 96 < mA ? sA[96] : 0.0f; y3 = 96 < mB ? sB[96] : 0.0f;
            x4 = 128 < mA ? sA[128] : 0.0f; y4 = 128 < mB ? sB[128] : 0.0f;
          }
          if (MULT && p.mult[b] != nullptr) {
            // layer-homogeneous form: a row stands for m_k identical kernels; the
            // multiplicities are read from global memory (they are shared by all specs)
            // multiplicities of rows begA.. / begB..: the staged copy (shared memory) or the global array
            const int32_t* mrow = (STAGED && mstaged) ? smult + mbase[b] : p.mult[b];
            const int32_t* mA = mrow + begA + lane;
            const int32_t* mB = mrow + begB + lane;
            int ka = 0, kb = 0;
            float pa = 0.0f, pb = 0.0f;
            const float xs[5] = {x0, x1, x2, x3, x4}, ys[5] = {y0, y1, y2, y3, y4};
#pragma unroll
            for (int r = 0; r < 5; ++r) {
              const int ma = 32 * r < mA_n(nA, lane) ? mA[32 * r] : 0;
              const int mb = 32 * r < mA_n(nB, lane) ? mB[32 * r] : 0;
              pa = fmaf((float)ma, xs[r], pa); ka += ma;
              pb = fmaf((float)mb, ys[r], pb); kb += mb;
            }
            for (int k = lane + 160; k < nA; k += 32) { const int m = mrow[begA + k]; pa = fmaf((float)m, (sA - lane)[k], pa); ka += m; }
            for (int k = lane + 160; k < nB; k += 32) { const int m = mrow[begB + k]; pb = fmaf((float)m, (sB - lane)[k], pb); kb += m; }
            accA += pa; accB += pb;
            cntA += ka; cntB += kb;                   // per-lane partial launch counts, summed with the shuffle tree below
          } else {
            accA += ((x0 + x1) + (x2 + x3)) + x4;
            accB += ((y0 + y1) + (y2 + y3)) + y4;
            if (nA > 160) accA += lane_tail(sA - lane, nA, lane);
            if (nB > 160) accB += lane_tail(sB - lane, nB, lane);
            if (!MULT || lane == 0) { cntA += nA; cntB += nB; }
          }
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        accA += __shfl_xor_sync(0xffffffffu, accA, o);
        accB += __shfl_xor_sync(0xffffffffu, accB, o);
        if (MULT) {
          cntA += __shfl_xor_sync(0xffffffffu, cntA, o);
          cntB += __shfl_xor_sync(0xffffffffu, cntB, o);
        }
      }
      if (lane < 2 && (lane == 0 || hasB)) {
        const float t_gpu = p.sp.body_scale * (lane == 0 ? accA : accB);
        const int count = lane == 0 ? cntA : cntB;
        // Eq. 4: t_step = max(t_gpu + n c_disp, l) + max(0, c_ovl - t_gpu) + c_tail
        const float t = fmaxf(fmaf((float)count, p.sp.c_disp, t_gpu), p.sp.floor_l) +
                        fmaxf(0.0f, p.sp.c_ovl - t_gpu) + p.sp.c_tail;
        p.step_lat[(long long)spec * p.n_steps + s0 + (lane == 0 ? jA : jB)] = t;
      }
    }
  };
  // Staged chunks of the unweighted large-problem instance: EIGHT LANES PER STEP (a warp sums four steps at once)
  // reading aligned 16-byte groups.  A step's elements [P, Q) of a bucket cover the groups [P / 4, ceil(Q / 4)):
  // the first and the last group are read by lanes 0 and 1 with per-element masks, the groups in between by all
  // eight lanes without any mask — one LDS.128 and three packed/scalar adds per four elements instead of a load,
  // a compare, a select and an add per element (the per-step instruction count drops from ~220 to ~45, which is
  // what kept this kernel at 59 % of the copy rate).  Fixed order: bit-reproducible.
  auto reduce_wide = [&]() {
    const int sub = lane >> 3, l8 = lane & 7;
    const float4* __restrict__ s4 = reinterpret_cast<const float4*>(sdata);
#pragma unroll 1
    for (int j = warp * 4 + sub; j < KS; j += kWarps * 4) {
      const bool valid = j < ns;
      float acc = 0.0f;
      int cnt = 0;
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        if (b < p.n_batches) {
          const int beg = valid ? offs[b][j] : 0, end = valid ? offs[b][j + 1] : 0;
          const int P = sbase[b] + beg, Q = sbase[b] + end;
          cnt += end - beg;
          if (Q > P) {
            const int G0 = P >> 2, G1 = (Q + 3) >> 2;
            float a0 = 0.0f, a1 = 0.0f, a2 = 0.0f, a3 = 0.0f;
#pragma unroll 1
            for (int g = G0 + 1 + l8; g < G1 - 1; g += 8) {
              const float4 v = s4[g];
              ks_add2(a0, a1, a0, a1, v.x, v.y);
              ks_add2(a2, a3, a2, a3, v.z, v.w);
            }
            if (l8 == 0 || (l8 == 1 && G1 - 1 > G0)) {
              const int g = l8 == 0 ? G0 : G1 - 1, e0 = 4 * g;
              const float4 v = s4[g];
              a0 += (e0 >= P && e0 < Q) ? v.x : 0.0f;
              a1 += (e0 + 1 >= P && e0 + 1 < Q) ? v.y : 0.0f;
              a2 += (e0 + 2 >= P && e0 + 2 < Q) ? v.z : 0.0f;
              a3 += (e0 + 3 >= P && e0 + 3 < Q) ? v.w : 0.0f;
            }
            acc += (a0 + a1) + (a2 + a3);
          }
        }
      }
      acc += __shfl_xor_sync(0xffffffffu, acc, 4);
      acc += __shfl_xor_sync(0xffffffffu, acc, 2);
      acc += __shfl_xor_sync(0xffffffffu, acc, 1);
      if (l8 == 0 && valid) {
        const float t_gpu = p.sp.body_scale * acc;
        // Eq. 4: t_step = max(t_gpu + n c_disp, l) + max(0, c_ovl - t_gpu) + c_tail
        const float t = fmaxf(fmaf((float)cnt, p.sp.c_disp, t_gpu), p.sp.floor_l) +
                        fmaxf(0.0f, p.sp.c_ovl - t_gpu) + p.sp.c_tail;
        p.step_lat[(long long)spec * p.n_steps + s0 + j] = t;
      }
    }
  };
  if (staged && !MULT && KS == kS) reduce_wide();
  else if (staged) reduce_all(std::true_type{});
  else reduce_all(std::false_type{});
}

constexpr int kTotThreads = 1024;

// One CTA per (spec, configuration): 1024 threads, four independent loads in flight per thread (the launch is a
// latency chain behind the step kernel: a 256-thread CTA walking its ~1,500 steps six dependent loads deep cost 5 us).
__global__ void __launch_bounds__(kTotThreads)
ks_cfg_total_kernel(const __grid_constant__ KsComposeParams p) {
  const int cfg = blockIdx.x % p.n_cfg;
  const int spec = blockIdx.x / p.n_cfg;
  // launched with programmatic stream serialization: everything above overlaps the tail of the step
  // kernel; nothing the stream produced before (step latencies, a caller's cfg_off) is read before this
  cudaGridDependencySynchronize();
  const int beg = __ldg(p.cfg_off + cfg), end = __ldg(p.cfg_off + cfg + 1);
  const float* sl = p.step_lat + (long long)spec * p.n_steps;
  double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
  int s = beg + (int)threadIdx.x;
  for (; s + 3 * kTotThreads < end; s += 4 * kTotThreads) {
    const float x0 = sl[s], x1 = sl[s + kTotThreads], x2 = sl[s + 2 * kTotThreads], x3 = sl[s + 3 * kTotThreads];
    a0 += (double)x0; a1 += (double)x1; a2 += (double)x2; a3 += (double)x3;
  }
  for (; s < end; s += kTotThreads) a0 += (double)sl[s];
  double acc = (a0 + a1) + (a2 + a3);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  __shared__ double part[kTotThreads / 32];
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x < 32) {
    double t = part[threadIdx.x];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (threadIdx.x == 0) p.cfg_lat[(long long)spec * p.n_cfg + cfg] = (float)t;
  }
}

}  // namespace

cudaError_t ks_launch_compose(const KsComposeParams& p, int num_sms, cudaStream_t st, int* launches) {
  const long long total = (long long)p.n_specs * p.n_steps;
  if (total > 0) {
    // a cfg2-sized problem (thousands of steps) is a latency chain per CTA: 8-step chunks give four times
    // as many, lighter CTAs (measured 2.3 us off a 99.6 us cfg2 step); 100k-step problems keep 32-step chunks
    // ... unless 32-step chunks already give every SM two CTAs (cfg3: 16,384 steps of 256 rows = 512 chunks): then the
    // eight-lanes-per-step reduction of the large chunks wins (cfg3 step kernel 13.4 us with 8-step chunks)
    const bool small = total <= kSmallSteps && total / kS < 2ll * (num_sms > 0 ? num_sms : 148);
    const int ks = small ? kSmallS : kS;
    const long long n_chunks = (long long)((p.n_steps + ks - 1) / ks) * p.n_specs;
    if (n_chunks > 0x7fffffffll) return cudaErrorInvalidValue;
    bool weighted = false;
    for (int b = 0; b < p.n_batches; ++b) weighted = weighted || p.mult[b] != nullptr;
    void (*kern)(const KsComposeParams);
    if (small) {
      kern = p.n_batches <= 1 ? ks_compose_kernel<1, false, kSmallS> : p.n_batches == 2 ? ks_compose_kernel<2, false, kSmallS> :
             p.n_batches == 3 ? ks_compose_kernel<3, false, kSmallS> : p.n_batches == 4 ? ks_compose_kernel<4, false, kSmallS> :
                                                                                         ks_compose_kernel<8, false, kSmallS>;
      if (weighted) kern = p.n_batches <= 4 ? ks_compose_kernel<4, true, kSmallS> : ks_compose_kernel<8, true, kSmallS>;
    } else {
      kern = p.n_batches <= 1 ? ks_compose_kernel<1, false, kS> : p.n_batches == 2 ? ks_compose_kernel<2, false, kS> :
             p.n_batches == 3 ? ks_compose_kernel<3, false, kS> : p.n_batches == 4 ? ks_compose_kernel<4, false, kS> :
                                                                                     ks_compose_kernel<8, false, kS>;
      if (weighted) kern = p.n_batches <= 4 ? ks_compose_kernel<4, true, kS> : ks_compose_kernel<8, true, kS>;
    }
    // the staging buffer: 47 KiB (four CTAs per SM) unless an average chunk would not fit it (cfg5: ~395 rows per
    // step), then 72 KiB (three CTAs per SM) — a chunk that does not fit is summed from global memory, far slower
    long long rows = 0;
    for (int b = 0; b < p.n_batches; ++b) rows += p.spec_stride[b];
    const bool big = (double)rows / (double)p.n_steps * ks > 0.85 * kCapFloats;
    KsComposeParams q = p;
    q.cap_floats = big ? kCapFloatsBig : kCapFloats;
    const size_t smem = (size_t)(q.cap_floats + kSlackFloats) * 4;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)((kCapFloatsBig + kSlackFloats) * 4));
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)n_chunks);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, kern, q);
    if (e != cudaSuccess) return e;
    if (launches) *launches += 1;
  }
  return ks_launch_cfg_totals(p, st, total > 0, launches);
}

cudaError_t ks_launch_cfg_totals(const KsComposeParams& p, cudaStream_t st, bool after_ours, int* launches) {
  if (p.n_cfg > 0 && p.n_specs > 0 && p.cfg_lat) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(p.n_cfg * p.n_specs));
    cfg.blockDim = dim3(kTotThreads);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // hide this launch under the step kernel's tail
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = after_ours ? 1 : 0;              // (no preceding kernel of ours: plain launch)
    cudaError_t e = cudaLaunchKernelEx(&cfg, ks_cfg_total_kernel, p);
    if (e != cudaSuccess) return e;
    if (launches) *launches += 1;
  }
  return cudaSuccess;
}
