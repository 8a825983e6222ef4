// ks_compose.cu — S6/S7: segmented reduction of kernel latencies into per-step GPU bodies
// (PAPER.md:231), the host-overlap step formula (Eq. 4) and per-configuration totals.
//
// ks_compose_kernel: persistent warps, one PAIR of consecutive steps per warp and trip (rows of a
// bucket are step-sorted, so the pair is one contiguous range of every bucket's latency array).
// One load fetches all CSR bounds of the pair (lane 3b+i), and the bounds of the warp's NEXT pair
// are requested before the current one is summed, so the only exposed memory round trip per trip
// is the latency data itself.  Per bucket and step the lanes read consecutive elements: five
// streaming loads (at clamped addresses, masked afterwards) cover segments up to 160 kernels, and
// the loads of every bucket are issued before the first add; longer segments stream the rest.  One fixed-order shuffle tree
// per step, Eq. 4 epilogue.  No atomics: bit-reproducible.
// Measured alternatives (profiles/README.md): staging chunks of 16-32 steps through shared memory
// with 1-D TMA bulk copies (2-4 stages, with and without a dedicated producer warp) or cp.async
// sustains 2.4-3.6 TB/s chip-wide on this access pattern and was not faster.
// Config totals: one CTA per (spec, config), fp64 accumulation.
#include "ks_internal.h"

namespace {

constexpr int kWarps = 8;
constexpr int kThreads = kWarps * 32;

// this lane's share of src[0, n) beyond the first 160 elements (rare: very long steps)
KS_DEV float lane_tail(const float* __restrict__ src, int n, int lane) {
  float a0 = 0.0f, a1 = 0.0f;
  int k = lane + 160;
#pragma unroll 1
  for (; k + 32 < n; k += 64) { a0 += __ldcs(src + k); a1 += __ldcs(src + k + 32); }
  if (k < n) a0 += __ldcs(src + k);
  return a0 + a1;
}

// NB = compile-time bound on the bucket count (1-4: exact, or 8): the bucket loop is fully unrolled so the
// loads of every bucket are in flight before the first add
template <int NB>
__global__ void __launch_bounds__(kThreads, NB <= 4 ? 4 : 2)
ks_compose_kernel(const __grid_constant__ KsComposeParams p) {
  const int lane = threadIdx.x & 31;
  const unsigned wid = blockIdx.x * kWarps + (threadIdx.x >> 5), n_warps = gridDim.x * kWarps;
  const unsigned pps = (unsigned)(p.n_steps + 1) / 2u;             // step pairs per spec
  const unsigned n_pairs = pps * (unsigned)p.n_specs;              // < 2^31 (checked by the launcher)

  // CSR offsets of pair q: lane 3b + i holds step_off[b][2c + i], i = 0..2 (clamped to n_steps)
  auto load_offs = [&](unsigned q) -> int {
    if (q >= n_pairs || lane >= 3 * p.n_batches) return 0;
    const int b = lane / 3, i = lane - 3 * b;
    const int s = 2 * (int)(q % pps) + i;
    return __ldg(p.step_off[b] + (s < p.n_steps ? s : p.n_steps));
  };

  int offv = load_offs(wid);
  for (unsigned q = wid; q < n_pairs; q += n_warps) {
    const int offn = load_offs(q + n_warps);        // next pair's offsets: in flight under this pair's sums
    const unsigned spec = q / pps;
    const int sA = 2 * (int)(q - spec * pps);
    const bool hasB = sA + 1 < p.n_steps;
    float x[NB][5], y[NB][5];
    int nA[NB], nB[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      const int beg = __shfl_sync(0xffffffffu, offv, 3 * b);
      const int mid = __shfl_sync(0xffffffffu, offv, 3 * b + 1);
      const int end = __shfl_sync(0xffffffffu, offv, 3 * b + 2);
      const bool on = b < p.n_batches;
      nA[b] = on ? mid - beg : 0;
      nB[b] = on ? end - mid : 0;
      // unconditional loads at clamped (always valid) addresses; out-of-segment lanes are masked
      // after ALL loads have been issued, so nothing waits on a load in between
      const float* __restrict__ a = nA[b] > 0 ? p.lat[b] + ((long long)spec * p.spec_stride[b] + beg) : p.step_lat;
      const float* __restrict__ c = nB[b] > 0 ? p.lat[b] + ((long long)spec * p.spec_stride[b] + mid) : p.step_lat;
      const int lastA = nA[b] > 0 ? nA[b] - 1 : 0, lastB = nB[b] > 0 ? nB[b] - 1 : 0;
#pragma unroll
      for (int r = 0; r < 5; ++r) {
        x[b][r] = __ldcs(a + min(lane + 32 * r, lastA));
        y[b][r] = __ldcs(c + min(lane + 32 * r, lastB));
      }
    }
#pragma unroll
    for (int b = 0; b < NB; ++b) {
#pragma unroll
      for (int r = 0; r < 5; ++r) {
        x[b][r] = lane + 32 * r < nA[b] ? x[b][r] : 0.0f;
        y[b][r] = lane + 32 * r < nB[b] ? y[b][r] : 0.0f;
      }
    }
    float accA = 0.0f, accB = 0.0f;
    int cntA = 0, cntB = 0;
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      accA += ((x[b][0] + x[b][1]) + (x[b][2] + x[b][3])) + x[b][4];
      accB += ((y[b][0] + y[b][1]) + (y[b][2] + y[b][3])) + y[b][4];
      cntA += nA[b];
      cntB += nB[b];
      if (nA[b] > 160 || nB[b] > 160) {             // warp-uniform: long steps stream the rest
        const int beg = __shfl_sync(0xffffffffu, offv, 3 * b);
        const float* __restrict__ a = p.lat[b] + ((long long)spec * p.spec_stride[b] + beg);
        if (nA[b] > 160) accA += lane_tail(a, nA[b], lane);
        if (nB[b] > 160) accB += lane_tail(a + nA[b], nB[b], lane);
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      accA += __shfl_xor_sync(0xffffffffu, accA, o);
      accB += __shfl_xor_sync(0xffffffffu, accB, o);
    }
    if (lane < 2 && (lane == 0 || hasB)) {
      const float t_gpu = p.sp.body_scale * (lane == 0 ? accA : accB);
      const int count = lane == 0 ? cntA : cntB;
      // Eq. 4: t_step = max(t_gpu + n c_disp, l) + max(0, c_ovl - t_gpu) + c_tail
      const float t = fmaxf(fmaf((float)count, p.sp.c_disp, t_gpu), p.sp.floor_l) +
                      fmaxf(0.0f, p.sp.c_ovl - t_gpu) + p.sp.c_tail;
      p.step_lat[(long long)spec * p.n_steps + sA + lane] = t;
    }
    offv = offn;
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
  const long long total = (long long)p.n_specs * p.n_steps;
  if (total > 0) {
    const long long n_pairs = (long long)((p.n_steps + 1) / 2) * p.n_specs;
    auto kern = p.n_batches <= 1 ? ks_compose_kernel<1> : p.n_batches == 2 ? ks_compose_kernel<2> :
                p.n_batches == 3 ? ks_compose_kernel<3> : p.n_batches == 4 ? ks_compose_kernel<4> : ks_compose_kernel<8>;
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kThreads, 0);
    if (e != cudaSuccess) return e;
    long long blocks = (long long)num_sms * (per_sm > 0 ? per_sm : 1);   // persistent: exactly one resident wave
    const long long need = (n_pairs + kWarps - 1) / kWarps;
    if (blocks > need) blocks = need;
    if (n_pairs + blocks * kWarps > 0x7fffffffll) return cudaErrorInvalidValue;
    kern<<<(unsigned)blocks, kThreads, 0, st>>>(p);
    e = cudaGetLastError();
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
