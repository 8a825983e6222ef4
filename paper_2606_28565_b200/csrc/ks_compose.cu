// ks_compose.cu — S6/S7: segmented reduction of kernel latencies into per-step GPU bodies
// (PAPER.md:231), the host-overlap step formula (Eq. 4) and per-configuration totals.
//
// One warp per (spec, step): for every family bucket the warp streams its CSR segment with
// coalesced loads (4 independent accumulators per lane), then a fixed-order shuffle tree combines
// the lanes — no atomics, so results are bit-reproducible.  Config totals: one CTA per
// (spec, config), fp64 accumulation, fixed-order block reduction.
#include "ks_internal.h"

namespace {

constexpr int kWarpsPerBlock = 8;

__global__ void __launch_bounds__(kWarpsPerBlock * 32)
ks_compose_kernel(const __grid_constant__ KsComposeParams p) {
  const int lane = threadIdx.x & 31;
  const long long warp = (long long)blockIdx.x * kWarpsPerBlock + (threadIdx.x >> 5);
  const long long total = (long long)p.n_specs * p.n_steps;
  if (warp >= total) return;
  const int spec = (int)(warp / p.n_steps);
  const int step = (int)(warp - (long long)spec * p.n_steps);

  float a0 = 0.0f, a1 = 0.0f, a2 = 0.0f, a3 = 0.0f;
  int count = 0;
  for (int b = 0; b < p.n_batches; ++b) {
    const int beg = __ldg(p.step_off[b] + step);
    const int end = __ldg(p.step_off[b] + step + 1);
    count += end - beg;
    const float* __restrict__ lat = p.lat[b] + (long long)spec * p.spec_stride[b];
    int k = beg + lane;
    for (; k + 96 < end; k += 128) {
      a0 += __ldcs(lat + k);
      a1 += __ldcs(lat + k + 32);
      a2 += __ldcs(lat + k + 64);
      a3 += __ldcs(lat + k + 96);
    }
    for (; k < end; k += 32) a0 += __ldcs(lat + k);
  }
  float acc = (a0 + a1) + (a2 + a3);
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
