// ks_mlp.cu — Tier-A kernel for H = 256 (cfg5): descriptor decode -> roofline -> features ->
// per-family MLP head on the 5th-gen tensor cores (tcgen05.mma, bf16 x bf16 -> fp32 in TMEM) ->
// sigmoid -> latency, fused.  S1-S3, S4a, S5 of DESIGN.md §1.  PAPER.md:191 Eq. 2, :199-201.
// (H <= 128 runs the warp-specialized pipeline in ks_mlp_ws.cu; ks_launch_mlp dispatches.)
//
// One persistent CTA per SM holds one family's weights in shared memory (staged by 1-D TMA bulk
// copies as pre-built UMMA operand images) and walks a contiguous range of 128-row tiles; it
// reloads weights when its range crosses into the next family bucket.  The W2 image of H = 256 is
// 136 KiB, so a single A2 buffer fits: one "slot" (128 rows = the 128 TMEM lanes) served by two
// warpgroups that split the hidden columns in halves.  Per (tile, spec):
//   WG0: decode + features -> bf16 A1 operand in smem        (A1 aliases the first K chunks of A2)
//   MMA1  D1[128 x H] = A1[128 x K1] . W1                    (bias b1 rides on two constant-1 feature columns)
//   epi1  D1 -> regs (tcgen05.ld) -> 2 GELU -> bf16 -> A2 smem, in 32-column chunks; after every chunk
//         the finished K range of MMA2 is issued, so layer 2 runs on the tensor core while the
//         ALUs are still activating the rest of layer 1
//   MMA2  D2[128 x H] = A2[128 x H] . W2/2  (+ one K=16 step: ones-block x {b2_hi, b2_lo})
//   epi2  D2 -> regs -> 2 GELU -> dot with w3/2 (fp32) -> z -> e = sigmoid(z) -> t = max(t_roof / e, t0)
// (The Cfg template also describes a four-slot layout with D2 aliasing D1 for H <= 128; it is kept
// compiled-out as the measured predecessor of the warp-specialized kernel: 115 us vs 100 us on cfg2.)
//
// Operand layout (both A and B): K-major, no swizzle: [K/8][rows][8] bf16, i.e. each 8-row x 16-byte
// core matrix is 128 contiguous bytes; SBO = 128 B, LBO = rows * 16 B.  A thread owns one row, so a
// warp's 16-byte stores to one K chunk cover 512 contiguous bytes (bank-conflict free).
#include "ks_mlp_common.cuh"

namespace {

using namespace ksmlp;

template <int NIN, int H>
struct Cfg {
  static constexpr int K1 = NIN == 32 ? 32 : 16;
  static constexpr int BIAS_ROW = NIN == 32 ? 22 : NIN;   // features >= 22 are identically zero (Q2)
  // A slot = one 128-row tile in flight.  H <= 128: one warpgroup per slot (a thread owns a whole
  // row), D2 reuses D1's TMEM columns, four slots per CTA hide each other's MMA / barrier waits.
  // H == 256: the W2 image alone is 136 KiB, so only one A2 buffer fits: one slot, two warpgroups
  // splitting the columns, D1 and D2 separate so MMA2 starts under layer 1's activation work.
  static constexpr int G = H == 256 ? 2 : 1;              // warpgroups per slot
  static constexpr bool ALIAS = H != 256;                 // D2 aliases D1
  static constexpr int NSLOTS = H == 256 ? 1 : 4;
  static constexpr int SLOT_THREADS = G * 128;
  static constexpr int THREADS = NSLOTS * SLOT_THREADS;
  static constexpr int TMEM_PER_SLOT = ALIAS ? H : 2 * H;
  static constexpr int TMEM_COLS = NSLOTS * TMEM_PER_SLOT;   // 256 (H = 64) or 512
  static constexpr int W1_BYTES = K1 * H * 2;
  static constexpr int W2_BYTES = (H + 16) * H * 2;
  static constexpr int A2_BYTES = (H / 8) * kChunkBytes;
  static constexpr int ONES_BYTES = 2 * kChunkBytes;
  static constexpr int OFF_W1 = 0;
  static constexpr int OFF_W2 = OFF_W1 + W1_BYTES;
  static constexpr int OFF_ONES = OFF_W2 + W2_BYTES;
  static constexpr int OFF_A2 = OFF_ONES + ONES_BYTES;
  static constexpr int OFF_W3 = OFF_A2 + NSLOTS * A2_BYTES;
  static constexpr int OFF_ZP = OFF_W3 + H * 4;
  static constexpr int OFF_BAR = OFF_ZP + NSLOTS * kRows * 4;
  static constexpr int SMEM_BYTES = OFF_BAR + 128;
  static constexpr int WGCOLS = H / G;        // columns per warpgroup
  static constexpr int NCHUNK = WGCOLS / 32;  // 32-column chunks per warpgroup
};

template <int NIN, int H, int FAM>
KS_DEV void process_bucket(const KsMlpParams& p, const int b, const int t_lo, const int t_hi, unsigned char* smem,
                           const uint32_t tmem_base, uint32_t& ph1, uint32_t& ph2) {
  using C = Cfg<NIN, H>;
  constexpr int NC = NCols<FAM>::v;
  const int tid = threadIdx.x;
  const int slot = tid / C::SLOT_THREADS;
  const int st = tid - slot * C::SLOT_THREADS;
  const int wg = st >> 7;
  const int r = st & 127;
  const KsBucketDev& bk = p.bk[b];

  unsigned char* A2 = smem + C::OFF_A2 + slot * C::A2_BYTES;
  const float* sw3 = reinterpret_cast<const float*>(smem + C::OFF_W3);
  float* zpart = reinterpret_cast<float*>(smem + C::OFF_ZP) + slot * kRows;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* mbar1 = bars + 1 + 2 * slot;
  uint64_t* mbar2 = bars + 2 + 2 * slot;

  const uint32_t a2_addr = ks_smem_u32(A2);
  const uint32_t w1_addr = ks_smem_u32(smem + C::OFF_W1);
  const uint32_t w2_addr = ks_smem_u32(smem + C::OFF_W2);
  const uint32_t ones_addr = ks_smem_u32(smem + C::OFF_ONES);
  const uint32_t d1 = tmem_base + (uint32_t)(slot * C::TMEM_PER_SLOT);
  const uint32_t d2 = C::ALIAS ? d1 : d1 + (uint32_t)H;
  const uint32_t lane_off = (uint32_t)((r >> 5) * 32) << 16;     // this warp's TMEM lane quarter
  constexpr uint32_t idesc = ks_umma_idesc_bf16(128, H);
  constexpr uint32_t B_LBO = H * 16;                              // K-chunk stride of a weight image
  const uint32_t bar_id = 1 + slot;
  const float b3 = p.head[b].b3;
  const int gelu_mode = p.gelu_mode;
  const int tile0 = p.tile_begin[b];
  const bool f32cols = bk.col_f32 != 0;

  // descriptor columns of the first tile; every later tile is prefetched one iteration ahead
  int vn[NC];
  {
    const int row = (t_lo + slot - tile0) * kRows + r;
    const bool ok = wg == 0 && t_lo + slot < t_hi && row < bk.n;
#pragma unroll
    for (int c = 0; c < NC; ++c) vn[c] = ok ? load_col_raw(bk.cols[c], row) : 0;
  }

  for (int t = t_lo + slot; t < t_hi; t += C::NSLOTS) {
    const int row = (t - tile0) * kRows + r;
    const bool valid = row < bk.n;
    int v[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) v[c] = col_value(vn[c], f32cols);
    {
      const int tn = t + C::NSLOTS;
      const int rown = (tn - tile0) * kRows + r;
      const bool ok = wg == 0 && tn < t_hi && rown < bk.n;
#pragma unroll
      for (int c = 0; c < NC; ++c) vn[c] = ok ? load_col_raw(bk.cols[c], rown) : 0;
    }
    for (int s = 0; s < p.n_specs; ++s) {
      const KsSpecDev& sp = p.specs.s[s];
      float t_roof = 0.0f;
      if (wg == 0) {
        // ---- S1-S3: decode, roofline, features -> bf16 A1 row
        const KsWork w = ks_decode<FAM>(v, bk, sp);
        const KsRoof rf = ks_roofline(w, sp);
        t_roof = rf.t_roof;
        float x[C::K1];
        ks_features<FAM, (NIN == 32 ? 22 : NIN)>(v, bk, sp, w, rf, x);
#pragma unroll
        for (int i = (NIN == 32 ? 22 : NIN); i < C::K1; ++i) x[i] = 0.0f;
        x[C::BIAS_ROW] = 1.0f;          // multiplies the b1_hi row of the W1 image
        x[C::BIAS_ROW + 1] = 1.0f;      // multiplies the b1_lo row
#pragma unroll
        for (int kc = 0; kc < C::K1 / 8; ++kc) {
          uint4 q;
          q.x = ks_pack_bf16x2(x[kc * 8 + 0], x[kc * 8 + 1]);
          q.y = ks_pack_bf16x2(x[kc * 8 + 2], x[kc * 8 + 3]);
          q.z = ks_pack_bf16x2(x[kc * 8 + 4], x[kc * 8 + 5]);
          q.w = ks_pack_bf16x2(x[kc * 8 + 6], x[kc * 8 + 7]);
          *reinterpret_cast<uint4*>(A2 + kc * kChunkBytes + r * 16) = q;
        }
        if (valid) {
          const long long o = (long long)s * bk.n + row;
          if (bk.tiles) bk.tiles[o] = (int)w.B;
          if (bk.waves) bk.waves[o] = (int)rf.W;
          if (bk.troof) bk.troof[o] = rf.t_roof;
        }
        ks_fence_proxy_async();
      }
      ks_tc_fence_before();
      ks_bar_sync(bar_id, C::SLOT_THREADS);
      // ---- MMA1: D1 = A1 . W1   (one thread issues for the slot)
      if (st == 0) {
        ks_tc_fence_after();
#pragma unroll
        for (int k = 0; k < C::K1 / 16; ++k) {
          const uint64_t ad = ks_umma_desc(a2_addr + k * 2 * kChunkBytes, kChunkBytes, 128);
          const uint64_t bd = ks_umma_desc(w1_addr + k * 2 * B_LBO, B_LBO, 128);
          ks_umma_bf16(d1, ad, bd, idesc, k > 0 ? 1u : 0u);
        }
        ks_umma_commit(mbar1);
      }
      ks_mbar_wait(mbar1, ph1);
      ph1 ^= 1u;
      ks_tc_fence_after();

      // ---- epi1: GELU(D1) -> A2, chunk by chunk
#pragma unroll 1
      for (int c = 0; c < C::NCHUNK; ++c) {
        const int col0 = wg * C::WGCOLS + c * 32;
        uint32_t acc[32];
        ks_tmem_ld32(d1 + lane_off + (uint32_t)col0, acc);
        ks_tmem_ld_wait();
        uint32_t pk[16];
        if (gelu_mode == 0) {
#pragma unroll
          for (int j = 0; j < 16; ++j)
            pk[j] = ks_pack_bf16x2(gelu2_f32(__uint_as_float(acc[2 * j])), gelu2_f32(__uint_as_float(acc[2 * j + 1])));
        } else {
#pragma unroll
          for (int j = 0; j < 16; ++j)
            pk[j] = gelu2_bf16x2(__uint_as_float(acc[2 * j]), __uint_as_float(acc[2 * j + 1]));
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          uint4 q;
          q.x = pk[4 * j + 0]; q.y = pk[4 * j + 1]; q.z = pk[4 * j + 2]; q.w = pk[4 * j + 3];
          *reinterpret_cast<uint4*>(A2 + (col0 / 8 + j) * kChunkBytes + r * 16) = q;
        }
        if (!C::ALIAS) {
          // D2 is separate: issue the K range of MMA2 that both warpgroups just finished, so
          // layer 2 runs on the tensor core under the rest of layer 1's activation work
          ks_fence_proxy_async();
          ks_tc_fence_before();
          ks_bar_sync(bar_id, C::SLOT_THREADS);
          if (st == 0) {
            ks_tc_fence_after();
#pragma unroll
            for (int g = 0; g < C::G; ++g) {
#pragma unroll
              for (int kk = 0; kk < 2; ++kk) {
                const int k16 = (g * C::WGCOLS + c * 32) / 16 + kk;
                const uint64_t ad = ks_umma_desc(a2_addr + k16 * 2 * kChunkBytes, kChunkBytes, 128);
                const uint64_t bd = ks_umma_desc(w2_addr + k16 * 2 * B_LBO, B_LBO, 128);
                ks_umma_bf16(d2, ad, bd, idesc, (c > 0 || g > 0 || kk > 0) ? 1u : 0u);
              }
            }
            if (c == C::NCHUNK - 1) {            // bias step: ones-block x {b2_hi, b2_lo, 0...}
              const uint64_t ad = ks_umma_desc(ones_addr, kChunkBytes, 128);
              const uint64_t bd = ks_umma_desc(w2_addr + (H / 8) * B_LBO, B_LBO, 128);
              ks_umma_bf16(d2, ad, bd, idesc, 1u);
              ks_umma_commit(mbar2);
            }
          }
        }
      }
      if (C::ALIAS) {
        // D2 overwrites D1: every warp of the slot has drained its D1 reads (tcgen05.wait::ld above)
        ks_fence_proxy_async();
        ks_tc_fence_before();
        ks_bar_sync(bar_id, C::SLOT_THREADS);
        if (st == 0) {
          ks_tc_fence_after();
#pragma unroll
          for (int k16 = 0; k16 < H / 16; ++k16) {
            const uint64_t ad = ks_umma_desc(a2_addr + k16 * 2 * kChunkBytes, kChunkBytes, 128);
            const uint64_t bd = ks_umma_desc(w2_addr + k16 * 2 * B_LBO, B_LBO, 128);
            ks_umma_bf16(d2, ad, bd, idesc, k16 > 0 ? 1u : 0u);
          }
          const uint64_t ad = ks_umma_desc(ones_addr, kChunkBytes, 128);
          const uint64_t bd = ks_umma_desc(w2_addr + (H / 8) * B_LBO, B_LBO, 128);
          ks_umma_bf16(d2, ad, bd, idesc, 1u);
          ks_umma_commit(mbar2);
        }
      }
      ks_mbar_wait(mbar2, ph2);
      ph2 ^= 1u;
      ks_tc_fence_after();

      // ---- epi2: GELU(D2) . w3
      float zp = 0.0f;
#pragma unroll 1
      for (int c = 0; c < C::NCHUNK; ++c) {
        const int col0 = wg * C::WGCOLS + c * 32;
        uint32_t acc[32];
        ks_tmem_ld32(d2 + lane_off + (uint32_t)col0, acc);
        ks_tmem_ld_wait();
        if (gelu_mode == 0) {
#pragma unroll
          for (int j = 0; j < 32; j += 4) {
            const float4 w4 = *reinterpret_cast<const float4*>(sw3 + col0 + j);
            zp = fmaf(gelu2_f32(__uint_as_float(acc[j + 0])), w4.x, zp);
            zp = fmaf(gelu2_f32(__uint_as_float(acc[j + 1])), w4.y, zp);
            zp = fmaf(gelu2_f32(__uint_as_float(acc[j + 2])), w4.z, zp);
            zp = fmaf(gelu2_f32(__uint_as_float(acc[j + 3])), w4.w, zp);
          }
        } else {
#pragma unroll
          for (int j = 0; j < 32; j += 4) {
            const float4 w4 = *reinterpret_cast<const float4*>(sw3 + col0 + j);
            const uint32_t g0 = gelu2_bf16x2(__uint_as_float(acc[j + 0]), __uint_as_float(acc[j + 1]));
            const uint32_t g1 = gelu2_bf16x2(__uint_as_float(acc[j + 2]), __uint_as_float(acc[j + 3]));
            zp = fmaf(__uint_as_float(g0 << 16), w4.x, zp);
            zp = fmaf(__uint_as_float(g0 & 0xffff0000u), w4.y, zp);
            zp = fmaf(__uint_as_float(g1 << 16), w4.z, zp);
            zp = fmaf(__uint_as_float(g1 & 0xffff0000u), w4.w, zp);
          }
        }
      }
      if (C::G == 2) {
        if (wg == 1) zpart[r] = zp;
        ks_tc_fence_before();
        ks_bar_sync(bar_id, C::SLOT_THREADS);
        if (wg == 0) zp += zpart[r];
      }
      if (wg == 0 && valid) {
        const float z = zp + b3;
        // eta = 1/e = 1 + exp(-z), guarded at e >= 2^-10 (Q3); Eq. 2 floor after eta
        const float eta = fminf(1.0f + __expf(-z), 1024.0f);
        bk.lat[(long long)s * bk.n + row] = fmaxf(t_roof * eta, sp.t0);
      }
    }
  }
}

template <int NIN, int H>
__global__ void __launch_bounds__(Cfg<NIN, H>::THREADS, 1)
ks_mlp_kernel(const __grid_constant__ KsMlpParams p) {
  using C = Cfg<NIN, H>;
  extern __shared__ __align__(1024) unsigned char smem[];
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint64_t* wbar = bars;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 1 + 2 * C::NSLOTS);
  const int tid = threadIdx.x;

  if (tid == 0) {
    ks_mbar_init(wbar, 1);
    for (int s = 0; s < C::NSLOTS; ++s) { ks_mbar_init(bars + 1 + 2 * s, 1); ks_mbar_init(bars + 2 + 2 * s, 1); }
    ks_fence_mbar_init();
  }
  if (tid < 32) { ks_tmem_alloc(tmem_slot, C::TMEM_COLS); ks_tmem_relinquish(); }
  if (tid < 128) {   // constant ones-block: K chunk 0 = {1, 1, 0, ...} per row, K chunk 1 = 0
    *reinterpret_cast<uint4*>(smem + C::OFF_ONES + tid * 16) = make_uint4(0x3F803F80u, 0u, 0u, 0u);
    *reinterpret_cast<uint4*>(smem + C::OFF_ONES + kChunkBytes + tid * 16) = make_uint4(0u, 0u, 0u, 0u);
  }
  ks_fence_proxy_async();
  ks_tc_fence_before();
  __syncthreads();
  ks_tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  const long long total = p.tile_begin[p.n_buckets];
  const int t_lo = (int)((long long)blockIdx.x * total / gridDim.x);
  const int t_hi = (int)((long long)(blockIdx.x + 1) * total / gridDim.x);
  uint32_t wphase = 0, ph1 = 0, ph2 = 0;

  for (int b = 0; b < p.n_buckets; ++b) {
    const int lo = t_lo > p.tile_begin[b] ? t_lo : p.tile_begin[b];
    const int hi = t_hi < p.tile_begin[b + 1] ? t_hi : p.tile_begin[b + 1];
    if (lo >= hi) continue;
    __syncthreads();                       // previous family's weights are no longer in use
    if (tid == 0) {                        // TMA-stage this family's operand images
      ks_mbar_expect_tx(wbar, (uint32_t)(C::W1_BYTES + C::W2_BYTES));
      ks_bulk_g2s(smem + C::OFF_W1, p.head[b].w1_img, C::W1_BYTES, wbar);
      for (int off = 0; off < C::W2_BYTES; off += 32768) {
        const int len = C::W2_BYTES - off < 32768 ? C::W2_BYTES - off : 32768;
        ks_bulk_g2s(smem + C::OFF_W2 + off, reinterpret_cast<const char*>(p.head[b].w2_img) + off, len, wbar);
      }
    }
    if (tid < H) reinterpret_cast<float*>(smem + C::OFF_W3)[tid] = __ldg(p.head[b].w3 + tid);
    __syncthreads();
    ks_mbar_wait(wbar, wphase);
    wphase ^= 1u;
    switch (p.bk[b].family) {
      case KS_FAM_GEMM: process_bucket<NIN, H, KS_FAM_GEMM>(p, b, lo, hi, smem, tmem_base, ph1, ph2); break;
      case KS_FAM_GROUPED_GEMM:
        process_bucket<NIN, H, KS_FAM_GROUPED_GEMM>(p, b, lo, hi, smem, tmem_base, ph1, ph2);
        break;
      case KS_FAM_ATTN: process_bucket<NIN, H, KS_FAM_ATTN>(p, b, lo, hi, smem, tmem_base, ph1, ph2); break;
      default: process_bucket<NIN, H, KS_FAM_ELEMWISE>(p, b, lo, hi, smem, tmem_base, ph1, ph2); break;
    }
  }
  ks_tc_fence_before();
  __syncthreads();
  if (tid < 32) ks_tmem_dealloc(tmem_base, C::TMEM_COLS);
}

template <int NIN, int H>
cudaError_t launch(const KsMlpParams& p, int num_sms, cudaStream_t st) {
  using C = Cfg<NIN, H>;
  const int total = p.tile_begin[p.n_buckets];
  if (total <= 0) return cudaSuccess;
  int grid = (total + C::NSLOTS - 1) / C::NSLOTS;
  if (grid > num_sms) grid = num_sms;
  auto kern = ks_mlp_kernel<NIN, H>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  kern<<<grid, C::THREADS, C::SMEM_BYTES, st>>>(p);
  return cudaGetLastError();
}

}  // namespace

int ks_mlp_k1(int n_in) { return n_in == 32 ? 32 : 16; }
size_t ks_mlp_w1_img_bytes(int n_in, int h) { return (size_t)ks_mlp_k1(n_in) * h * 2; }
size_t ks_mlp_w2_img_bytes(int h) { return (size_t)(h + 16) * h * 2; }

cudaError_t ks_launch_mlp(const KsMlpParams& p, int n_in, int h, int num_sms, cudaStream_t st) {
#define KS_CASE(NI, HH) \
  if (n_in == NI && h == HH) return launch<NI, HH>(p, num_sms, st);
  if (h <= 128) return ks_launch_mlp_ws(p, n_in, h, num_sms, st);   // warp-specialized pipeline (ks_mlp_ws.cu)
  if (h == 256 && p.gelu_mode < 2) return ks_launch_mlp_ws256(p, n_in, num_sms, st);   // ks_mlp_ws256.cu
  KS_CASE(8, 256) KS_CASE(12, 256) KS_CASE(32, 256)
#undef KS_CASE
  return cudaErrorInvalidValue;
}
