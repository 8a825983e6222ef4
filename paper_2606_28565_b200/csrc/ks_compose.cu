// ks_compose.cu — S6/S7: segmented reduction of kernel latencies into per-step GPU bodies
// (PAPER.md:231), the host-overlap step formula (Eq. 4) and per-configuration totals.
//
// One warp per (spec, step): one parallel load fetches every bucket's CSR bounds, then the first
// 128 elements of every bucket are loaded before the first add (one memory round trip per step),
// longer segments stream the rest; a fixed-order shuffle tree combines the lanes — no atomics, so results are bit-reproducible.  Config totals: one CTA per
// (spec, config), fp64 accumulation, fixed-order block reduction.
#include "ks_internal.h"

namespace {

constexpr int kWarpsPerBlock = 8;

constexpr int kRounds = 4;   // predicated first-round loads per bucket issued before any add

__global__ void __launch_bounds__(kWarpsPerBlock * 32)
ks_compose_kernel(const __grid_constant__ KsComposeParams p) {
  const int lane = threadIdx.x & 31;
  const long long warp = (long long)blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  const long long total = (long long)p.n_specs * p.n_steps;
  if (warp >= total) return;
  const int spec = (int)(warp / p.n_steps);
  const int step = (int)(warp - (long long)spec * p.n_steps);

  // all CSR offsets of this step in ONE parallel load: lane 2b -> begin, lane 2b+1 -> end of bucket b
  int off = 0;
  if (lane < 2 * p.n_batches) off = __ldg(p.step_off[lane >> 1] + step + (lane & 1));

  // first kRounds x 32 elements of every bucket: issue every load before the first add so one
  // memory round trip covers the whole step for typical segment lengths (<= 128 per bucket)
  float x[KS_MAX_BATCHES][kRounds];
  int count = 0;
#pragma unroll
  for (int b = 0; b < KS_MAX_BATCHES; ++b) {
    const int beg = __shfl_sync(0xffffffffu, off, 2 * b);
    const int end = __shfl_sync(0xffffffffu, off, 2 * b + 1);
    const bool on = b < p.n_batches;
    count += on ? end - beg : 0;
    const float* __restrict__ lat = p.lat[b] + (long long)spec * p.spec_stride[b];
#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
      const int k = beg + lane + 32 * r;
      x[b][r] = (on && k < end) ? __ldcs(lat + k) : 0.0f;
    }
  }
  float a[kRounds];
#pragma unroll
  for (int r = 0; r < kRounds; ++r) a[r] = 0.0f;
#pragma unroll
  for (int b = 0; b < KS_MAX_BATCHES; ++b)
#pragma unroll
    for (int r = 0; r < kRounds; ++r) a[r] += x[b][r];
  // long segments: stream the remainder
  for (int b = 0; b < p.n_batches; ++b) {
    const int beg = __shfl_sync(0xffffffffu, off, 2 * b);
    const int end = __shfl_sync(0xffffffffu, off, 2 * b + 1);
    if (end - beg <= 32 * kRounds) continue;
    const float* __restrict__ lat = p.lat[b] + (long long)spec * p.spec_stride[b];
    int k = beg + lane + 32 * kRounds;
    for (; k + 96 < end; k += 128) {
      a[0] += __ldcs(lat + k);
      a[1] += __ldcs(lat + k + 32);
      a[2] += __ldcs(lat + k + 64);
      a[3] += __ldcs(lat + k + 96);
    }
    for (; k < end; k += 32) a[0] += __ldcs(lat + k);
  }
  float acc = (a[0] + a[1]) + (a[2] + a[3]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) {
    const float t_gpu = p.sp.body_scale * acc;
    // Eq. 4: t_step = max(t_gpu + n c_disp, l) + max(0, c_ovl - t_gpu) + c_tail
    const float t = fmaxf(fmaf((float)count, p.sp.c_disp, t_gpu), p.sp.floor_l) +
                    fmaxf(0.0f, p.sp.c_ovl - t_gpu) + p.sp.c_tail;
    p.step_lat[(long long)spec * p.n_steps + step] = t;
  }
}

__global__ void __launch_bounds__(256)
ks_cfg_total_kernel(const __grid_constant__ KsComposeParams p) {
  const int cfg = blockIdx.x % p.n_cfg;
  const int spec = blockIdx.x / p.n_cfg;
  const int beg = __ldg(p.cfg_off + cfg), end = __ldg(p.cfg_off + cfg + 1);
  const float* __restrict__ sl = p.step_lat + (long long)spec * p.n_steps;
  double acc = 0.0;
  for (int s = beg + threadIdx.x; s < end; s += blockDim.x) acc += (double)sl[s];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  __shared__ double part[8];
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += part[w];
    p.cfg_lat[(long long)spec * p.n_cfg + cfg] = (float)t;
  }
}

}  // namespace

cudaError_t ks_launch_compose(const KsComposeParams& p, int num_sms, cudaStream_t st, int* launches) {
  (void)num_sms;
  const long long total = (long long)p.n_specs * p.n_steps;
  if (total > 0) {
    const long long blocks = (total + kWarpsPerBlock - 1) / kWarpsPerBlock;
    if (blocks > 0x7fffffffll) return cudaErrorInvalidValue;
    ks_compose_kernel<<<(unsigned)blocks, kWarpsPerBlock * 32, 0, st>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (launches) *launches += 1;
  }
  if (p.n_cfg > 0 && p.n_specs > 0 && p.cfg_lat) {
    ks_cfg_total_kernel<<<(unsigned)(p.n_cfg * p.n_specs), 256, 0, st>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (launches) *launches += 1;
  }
  return cudaSuccess;
}
