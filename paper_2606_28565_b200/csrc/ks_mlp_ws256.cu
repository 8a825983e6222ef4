// ks_mlp_ws256.cu — Tier-A kernel for H = 256 (cfg5, the what-if sweep): the warp-specialized
// tcgen05 pipeline of ks_mlp_ws.cu re-laid-out for a head whose W2 image alone is 128 KiB.
// S1-S3, S4a, S5 of DESIGN.md §1 (PAPER.md:191 Eq. 2, :199-201 per-family heads), fused.
//
// Shared memory holds W1, W2 (without bias rows), ONE A1 and ONE A2 buffer (225-229 KB in all) and TMEM
// holds one D1 and one D2 (256 + 256 columns), so nothing is double-buffered by item; instead the
// hand-over between layer 1 and layer 2 is pipelined at the granularity of 64-column K groups:
//   warps 0-3    PRODUCER  thread = row: decode + roofline + features -> bf16 A1 (after MMA1 of the
//                          previous item has consumed it), t_roof -> 4-deep ring
//   warps 4-11   EPI1      warpgroup g activates D1 columns [128 g, 128 g + 128): tcgen05.ld 16 columns
//                          (double-buffered) -> 2 GELU -> bf16 -> A2 K groups 2g, 2g+1; group k of item
//                          q is stored once MMA2(q-1) has consumed group k (a2_free[k]) and announced
//                          on a2_full[k]; d1_free as soon as the last D1 column is in registers
//   warp  20     MMA       MMA2(q) is issued group by group as the groups arrive (order 0, 2, 1, 3),
//                          with MMA1(q+1) slotted in as soon as D1 is drained: layer 2 of item q runs
//                          on the tensor core under the rest of layer 1's activation work, and layer 1
//                          of item q+1 is ready when EPI1 finishes item q
//   warps 12-19  EPI2      both warpgroups take 64 columns of D2 half 0, then 64 columns of half 1 (warpgroup g: columns
//                          [64 g, 64 g + 64) and [128 + 64 g, 128 + 64 g + 64)): (+ b2 in fp32 unless n_in = 32) -> 2 GELU -> dot with w3/2;
//                          while they are on one half the tensor core refills the other with the next item (a clock64
//                          trace showed the item period = activation of a half + its refill when a warpgroup owned a
//                          whole half).  Ensembles keep a half per warpgroup (a member's columns stay in one warpgroup).
//                          The two partial dots meet in shared memory; sigmoid, latency
// so EPI1(q+1) and EPI2(q) share the MUFU pipe while the tensor core works on both items.
// b2: in the H <= 128 kernels it rides through the tensor core as one more K step against a ones-block; there is no
// room for that here (12 KiB).  n_in = 32 (cfg5) gets it through the tensor core all the same: a 4 KiB bias chunk in
// front of the W2 image and A1's own constant-1 columns as the A operand (Cfg256::BIAS_MMA); other widths add it in
// the fp32 epilogue.
// Every mbarrier completes exactly once per item, so its phase parity is q & 1; a waiter for item q
// always runs before the completion for item q+1 can happen (that one depends on the waiter).
#include <type_traits>
#include "ks_mlp_common.cuh"

namespace {

using namespace ksmlp;

constexpr int H = 256;
constexpr int kProducerWarps = 4, kEpiWarps = 8;
constexpr int kThreads = (kProducerWarps + 2 * kEpiWarps + 1) * 32;   // 672
constexpr int kMmaWarp = kProducerWarps + 2 * kEpiWarps;
constexpr int kRing = 4;
constexpr int kGroups = 4;                         // A2 K groups of 64 columns

template <int NIN>
struct Cfg256 {
  static constexpr int K1 = NIN == 32 ? 32 : 16;
  static constexpr int BIAS_ROW = NIN == 32 ? 22 : NIN;
  static constexpr int W1_BYTES = K1 * H * 2;
  static constexpr int W2_BYTES = H * H * 2;       // K rows 0..H-1 of the image: the bias rows are not staged
  static constexpr int A1_BYTES = (K1 / 8) * kChunkBytes;
  static constexpr int A2_BYTES = (H / 8) * kChunkBytes;
  static constexpr int OFF_W1 = 0;
  static constexpr int OFF_B2IMG = OFF_W1 + W1_BYTES;         // directly in front of the W2 image (see BIAS_MMA below)
  static constexpr int OFF_W2 = OFF_B2IMG + (NIN == 32 ? H * 16 : 0);
  static constexpr int OFF_A1 = OFF_W2 + W2_BYTES;
  static constexpr int OFF_A2 = OFF_A1 + A1_BYTES;
  static constexpr int OFF_W3 = OFF_A2 + A2_BYTES;            // [H] fp32 w3/2 of the current family
  static constexpr int OFF_B2 = OFF_W3 + H * 4;               // [H] fp32 b2
  static constexpr int OFF_RING = OFF_B2 + H * 4;             // [kRing][128] fp32 t_roof
  static constexpr int OFF_ZP = OFF_RING + kRing * kRows * 4; // [2][128] fp32 partial dots of warpgroup 1
  // b2 through the tensor core (NIN = 32 only): one K chunk [H][8] bf16 with b2 hi / lo at positions 6, 7 -- where A1
  // carries layer 1's constant-1 columns 22, 23 -- as the FIRST K chunk of a K = 16 MMA against A1 chunks 2, 3 (columns
  // 16..31: six features that meet zero rows, the two ones, then eight zero columns); the second K chunk the MMA reads
  // is whatever follows in shared memory, the first chunk of the W2 image: finite values that meet A1's zero columns
  static constexpr bool BIAS_MMA = NIN == 32;
  static constexpr int B2IMG_BYTES = BIAS_MMA ? H * 16 : 0;
  static constexpr int OFF_BAR = OFF_ZP + 2 * kRows * 4;
  static constexpr int SMEM_BYTES = OFF_BAR + 256;   // 21 barriers + TMEM slot (192) + TileMap
  static_assert(SMEM_BYTES <= 232448, "shared memory");
};

// MMA2, D2_FREE, Z_FULL, Z_FREE come in pairs (column half of D2 / parity of the item)
enum { BAR_W = 0, BAR_DRAIN, BAR_A1_FULL, BAR_MMA1, BAR_D1_FREE, BAR_MMA2, BAR_D2_FREE = BAR_MMA2 + 2,
       BAR_Z_FULL = BAR_D2_FREE + 2, BAR_Z_FREE = BAR_Z_FULL + 2, BAR_A2_FULL = BAR_Z_FREE + 2,
       BAR_A2_FREE = BAR_A2_FULL + kGroups, BAR_COUNT = BAR_A2_FREE + kGroups };

struct Range { int lo, hi; };
KS_DEV Range bucket_range(const TileMap& tm, int b, int t_lo, int t_hi) {
  Range r;
  r.lo = t_lo > tm.tb[b] ? t_lo : tm.tb[b];
  r.hi = t_hi < tm.tb[b + 1] ? t_hi : tm.tb[b + 1];
  return r;
}

// ------------------------------------------------------------------ PRODUCER (warps 0-3)
template <int NIN, int FAM>
KS_DEV void producer_bucket(const KsMlpParams& p, const TileMap& tm, const int b, const Range tr, unsigned char* smem,
                            uint64_t* bars, uint32_t& q) {
  using C = Cfg256<NIN>;
  constexpr int NC = NCols<FAM>::v;
  const int r = threadIdx.x;
  const KsBucketDev& bk = p.bk[b];
  const int tile0 = tm.tb[b], ne = tm.ne[b];
  const bool f32cols = bk.col_f32 != 0;
  float* ring = reinterpret_cast<float*>(smem + C::OFF_RING);
  unsigned char* A1 = smem + C::OFF_A1;

  int vn[NC];
  int row_next;                                    // descriptor row whose columns sit in vn
  {
    const int pos = (tr.lo - tile0) * kRows + r;
    row_next = pos < ne ? map_row(bk, pos) : 0;
#pragma unroll
    for (int c = 0; c < NC; ++c) vn[c] = pos < ne ? load_col_raw(bk.cols[c], row_next) : 0;
  }
  for (int t = tr.lo; t < tr.hi; ++t) {
    const int pos = (t - tile0) * kRows + r;
    const bool valid = pos < ne;
    const int row = row_next;                        // descriptor row of this list position
    int v[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) v[c] = col_value(vn[c], f32cols);
    {
      const bool ok = t + 1 < tr.hi && pos + kRows < ne;
      row_next = ok ? map_row(bk, pos + kRows) : 0;
#pragma unroll
      for (int c = 0; c < NC; ++c) vn[c] = ok ? load_col_raw(bk.cols[c], row_next) : 0;
    }
    for (int s = 0; s < p.n_specs; ++s, ++q) {
      const KsSpecDev& sp = p.specs.s[s];
      uint4 a1[C::K1 / 8];
      KsWork w;
      KsRoof rf;
      const float t_roof = feature_row<FAM, NIN, C::K1, C::BIAS_ROW>(v, bk, sp, a1, w, rf);
      if (valid) {
        const long long o = (long long)s * bk.n + row;
        if (bk.tiles) bk.tiles[o] = (int)w.B;
        if (bk.waves) bk.waves[o] = (int)rf.W;
        if (bk.troof) bk.troof[o] = rf.t_roof;
      }
      if (q >= 1u) ks_mbar_wait(bars + BAR_MMA1, (q - 1u) & 1u);    // MMA1(q-1) has consumed A1
#pragma unroll
      for (int kc = 0; kc < C::K1 / 8; ++kc) *reinterpret_cast<uint4*>(A1 + kc * kChunkBytes + r * 16) = a1[kc];
      // ring slot q & 3 was last used by item q-4; EPI2 finished it before MMA1(q-1) could be issued
      ring[(q & (kRing - 1)) * kRows + r] = t_roof;
      ks_fence_proxy_async();
      ks_mbar_arrive(bars + BAR_A1_FULL);
    }
  }
}

// ------------------------------------------------------------------ EPI1 (warps 4-11)
template <int NIN, int GM>
KS_DEV void epi1_items(const KsMlpParams& p, const uint32_t n_items, unsigned char* smem, uint64_t* bars,
                       const uint32_t tmem_base) {
  using C = Cfg256<NIN>;
  const int e = threadIdx.x - kProducerWarps * 32;
  const int wg = e >> 7;                                            // columns [128 wg, 128 wg + 128)
  const int r = e & 127;
  const uint32_t lane_off = (uint32_t)((r >> 5) * 32) << 16;
  unsigned char* A2 = smem + C::OFF_A2;
  const uint32_t d1 = tmem_base + lane_off + (uint32_t)(wg * 128);
  // c16: 16-column sub-chunk within the warpgroup's half; wait_bar: the K group's a2_free barrier when this
  // sub-chunk is the first of the group.  The wait sits between the arithmetic and the stores, so the GELUs of
  // a group's first sub-chunk run while layer 2 of the previous item still reads the group (2 % on cfg5).
  auto act_store = [&](const uint32_t* a, int c16, uint64_t* wait_bar, uint32_t wait_par) {
    uint32_t pk[8];
    if (GM == 0) {
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        float g0, g1;
        gelu2_f32x2(__uint_as_float(a[2 * j]), __uint_as_float(a[2 * j + 1]), g0, g1);
        pk[j] = ks_pack_bf16x2(g0, g1);
      }
    } else {
#pragma unroll
      for (int j = 0; j < 8; ++j) pk[j] = gelu2_bf16x2(__uint_as_float(a[2 * j]), __uint_as_float(a[2 * j + 1]));
    }
    if (wait_bar) ks_mbar_wait(wait_bar, wait_par);
    const int kc = wg * 16 + c16 * 2;                               // 8-column K chunk index
    *reinterpret_cast<uint4*>(A2 + (kc + 0) * kChunkBytes + r * 16) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
    *reinterpret_cast<uint4*>(A2 + (kc + 1) * kChunkBytes + r * 16) = make_uint4(pk[4], pk[5], pk[6], pk[7]);
  };
  for (uint32_t q = 0; q < n_items; ++q) {
    const uint32_t par = q & 1u;
    ks_mbar_wait(bars + BAR_MMA1, par);                             // D1 holds item q
    ks_tc_fence_after();
    uint32_t accA[16], accB[16];
    ks_tmem_ld16(d1, accA);
#pragma unroll 1
    for (int c = 0; c < 8; c += 2) {                                // 8 sub-chunks = 2 K groups of 64 columns
      ks_tmem_ld_wait();
      ks_tmem_ld16(d1 + (uint32_t)((c + 1) * 16), accB);
      act_store(accA, c, ((c & 3) == 0 && q >= 1u) ? bars + BAR_A2_FREE + wg * 2 + (c >> 2) : nullptr, par ^ 1u);
      ks_tmem_ld_wait();
      if (c + 2 < 8) {
        ks_tmem_ld16(d1 + (uint32_t)((c + 2) * 16), accA);
      } else {                                                      // D1 is drained: MMA1(q+1) may overwrite it
        ks_tc_fence_before();
        ks_mbar_arrive(bars + BAR_D1_FREE);
      }
      act_store(accB, c + 1, nullptr, 0u);
      if ((c & 3) == 2) {                                           // a K group of 64 columns is complete
        ks_fence_proxy_async();
        ks_mbar_arrive(bars + BAR_A2_FULL + wg * 2 + (c >> 2));
      }
    }
  }
}

// ------------------------------------------------------------------ EPI2 (warps 12-19)
template <int NIN, int GM, bool ENS>
KS_DEV void epi2_all(const KsMlpParams& p, const TileMap& tm, const int t_lo, const int t_hi, unsigned char* smem,
                     uint64_t* bars, const uint32_t tmem_base) {
  using C = Cfg256<NIN>;
  const int e = threadIdx.x - (kProducerWarps + kEpiWarps) * 32;   // 0..255
  const int wg = e >> 7;
  const int r = e & 127;
  const uint32_t lane_off = (uint32_t)((r >> 5) * 32) << 16;
  const float* ring = reinterpret_cast<const float*>(smem + C::OFF_RING);
  float* sw3 = reinterpret_cast<float*>(smem + C::OFF_W3);
  float* sb2 = reinterpret_cast<float*>(smem + C::OFF_B2);
  float* zpart = reinterpret_cast<float*>(smem + C::OFF_ZP);
  const uint32_t d2 = tmem_base + (uint32_t)H + lane_off + (uint32_t)(wg * 128);
  uint32_t q = 0;
  for (int b = 0; b < p.n_buckets; ++b) {
    const Range tr = bucket_range(tm, b, t_lo, t_hi);
    if (tr.lo >= tr.hi) continue;
    const KsBucketDev& bk = p.bk[b];
    // this family's layer-3 weights and layer-2 bias: a warpgroup stages and reads only its own 128 columns
    ks_bar_sync(2 + wg, 128);
    {
      // ENS: the warpgroup owns columns [128 wg, 128 wg + 128); otherwise 64 columns of EACH half of D2:
      // [64 wg, 64 wg + 64) and [128 + 64 wg, 128 + 64 wg + 64)
      const int sc = ENS ? e : ((r >> 6) * 128 + wg * 64 + (r & 63));
      sw3[sc] = __ldg(p.head[b].w3 + sc);
      sb2[sc] = __ldg(p.head[b].b2 + sc);
    }
    ks_bar_sync(2 + wg, 128);
    const KsHeadDev& hd = p.head[b];
    const float b3 = hd.b3, out_sgn = hd.out_sgn, out_lo = hd.out_lo, out_add = hd.out_add;
    const int members = ENS ? hd.members : 1;                                  // > 1: MLP ensemble (2, 4 or 8 members here)
    const int ens_mask = members > 1 ? H / 16 / members - 1 : 0;     // chunks per member - 1 (member width 32 .. 128)
    const int tile0 = tm.tb[b], ne = tm.ne[b];
    // per-bucket parameters live in registers across the item loop (the asm keeps the compiler from
    // re-reading them with indexed constant loads between two items; see ks_mlp_ws.cu)
    const int* idx = bk.idx;
    float* lat = bk.lat;
    int bn = bk.n, n_specs = p.n_specs;
    asm volatile("" : "+l"(idx), "+l"(lat), "+r"(bn), "+r"(n_specs));
    for (int t = tr.lo; t < tr.hi; ++t) {
      const int pos = (t - tile0) * kRows + r;
      const bool valid = pos < ne;
      const int row = valid ? (idx ? __ldg(idx + pos) : pos) : 0;
      for (int s = 0; s < n_specs; ++s, ++q) {
        float z;
        if (ENS) {
          ks_mbar_wait(bars + BAR_MMA2 + wg, q & 1u);                 // this half of D2 holds item q
          ks_tc_fence_after();
          uint32_t accA[16], accB[16];
          ks_tmem_ld16(d2, accA);
          float z0 = 0.0f, z1 = 0.0f, z2 = 0.0f, z3 = 0.0f;
          auto act_dot = [&](const uint32_t* a, int c16) {
            const int col = wg * 128 + c16 * 16;
  #pragma unroll
            for (int j = 0; j < 16; j += 4) {
              const float4 w4 = *reinterpret_cast<const float4*>(sw3 + col + j);
              float x0, x1, x2, x3;
              if (C::BIAS_MMA) {
                x0 = __uint_as_float(a[j + 0]); x1 = __uint_as_float(a[j + 1]);
                x2 = __uint_as_float(a[j + 2]); x3 = __uint_as_float(a[j + 3]);
              } else {
                const float4 b4 = *reinterpret_cast<const float4*>(sb2 + col + j);
                ks_add2(x0, x1, __uint_as_float(a[j + 0]), __uint_as_float(a[j + 1]), b4.x, b4.y);
                ks_add2(x2, x3, __uint_as_float(a[j + 2]), __uint_as_float(a[j + 3]), b4.z, b4.w);
              }
              if (GM == 0) {
                float g0, g1, g2, g3;
                gelu2_f32x2(x0, x1, g0, g1);
                gelu2_f32x2(x2, x3, g2, g3);
                ks_fma2(z0, z1, g0, g1, w4.x, w4.y, z0, z1);
                ks_fma2(z2, z3, g2, g3, w4.z, w4.w, z2, z3);
              } else {
                const uint32_t g0 = gelu2_bf16x2(x0, x1), g1 = gelu2_bf16x2(x2, x3);
                z0 = fmaf(__uint_as_float(g0 << 16), w4.x, z0);
                z1 = fmaf(__uint_as_float(g0 & 0xffff0000u), w4.y, z1);
                z2 = fmaf(__uint_as_float(g1 << 16), w4.z, z2);
                z3 = fmaf(__uint_as_float(g1 & 0xffff0000u), w4.w, z3);
              }
            }
          };
          float esum = 0.0f;                         // ensemble: sum of this half's members' efficiencies
          auto sweep = [&](auto ens) {
            int m = wg * (members >> 1);             // first member of this warpgroup's 128 columns
  #pragma unroll 1
            for (int c = 0; c < 8; c += 2) {
              ks_tmem_ld_wait();
              ks_tmem_ld16(d2 + (uint32_t)((c + 1) * 16), accB);
              act_dot(accA, c);
              ks_tmem_ld_wait();
              if (c + 2 < 8) {
                ks_tmem_ld16(d2 + (uint32_t)((c + 2) * 16), accA);
              } else {                                                  // D2 is drained: MMA2(q+1) may overwrite it
                ks_tc_fence_before();
                ks_mbar_arrive(bars + BAR_D2_FREE + wg);
              }
              act_dot(accB, c + 1);
              if (decltype(ens)::value && ((c + 2) & ens_mask) == 0) {  // last column of member m (Q17)
                const float zm = ((z0 + z1) + (z2 + z3)) + hd.b3m[m++];
                esum += __fdividef(1.0f, 1.0f + __expf(-zm));
                z0 = z1 = z2 = z3 = 0.0f;
              }
            }
          };
          if (members > 1) sweep(std::true_type{}); else sweep(std::false_type{});
          // single head: partial logit of this half; ensemble: partial sum of efficiencies
          z = members > 1 ? esum : (z0 + z1) + (z2 + z3);
        } else {
          // Both warpgroups activate 64 columns of half 0, then 64 columns of half 1: while they are on half 1 the tensor
          // core refills half 0 with the next item and vice versa, so the 1,000-1,300 cycles of a refill no longer sit
          // between two activations of the same half (clock64 trace: the item period was activation + refill).
          float z0 = 0.0f, z1 = 0.0f, z2 = 0.0f, z3 = 0.0f;
#pragma unroll 1
          for (int h = 0; h < 2; ++h) {
            ks_mbar_wait(bars + BAR_MMA2 + h, q & 1u);               // half h of D2 holds item q
            ks_tc_fence_after();
            const uint32_t d2h = tmem_base + (uint32_t)H + lane_off + (uint32_t)(h * 128 + wg * 64);
            const int col0 = h * 128 + wg * 64;
            uint32_t accA[16], accB[16];
            ks_tmem_ld16(d2h, accA);
            auto act_dot = [&](const uint32_t* a, int c16) {
              const int col = col0 + c16 * 16;
#pragma unroll
              for (int j = 0; j < 16; j += 4) {
                const float4 w4 = *reinterpret_cast<const float4*>(sw3 + col + j);
                float x0, x1, x2, x3;
                if (C::BIAS_MMA) {
                  x0 = __uint_as_float(a[j + 0]); x1 = __uint_as_float(a[j + 1]);
                  x2 = __uint_as_float(a[j + 2]); x3 = __uint_as_float(a[j + 3]);
                } else {
                  const float4 b4 = *reinterpret_cast<const float4*>(sb2 + col + j);
                  ks_add2(x0, x1, __uint_as_float(a[j + 0]), __uint_as_float(a[j + 1]), b4.x, b4.y);
                  ks_add2(x2, x3, __uint_as_float(a[j + 2]), __uint_as_float(a[j + 3]), b4.z, b4.w);
                }
                if (GM == 0) {
                  float g0, g1, g2, g3;
                  gelu2_f32x2(x0, x1, g0, g1);
                  gelu2_f32x2(x2, x3, g2, g3);
                  ks_fma2(z0, z1, g0, g1, w4.x, w4.y, z0, z1);
                  ks_fma2(z2, z3, g2, g3, w4.z, w4.w, z2, z3);
                } else {
                  const uint32_t g0 = gelu2_bf16x2(x0, x1), g1 = gelu2_bf16x2(x2, x3);
                  z0 = fmaf(__uint_as_float(g0 << 16), w4.x, z0);
                  z1 = fmaf(__uint_as_float(g0 & 0xffff0000u), w4.y, z1);
                  z2 = fmaf(__uint_as_float(g1 << 16), w4.z, z2);
                  z3 = fmaf(__uint_as_float(g1 & 0xffff0000u), w4.w, z3);
                }
              }
            };
#pragma unroll 1
            for (int c = 0; c < 4; c += 2) {
              ks_tmem_ld_wait();
              ks_tmem_ld16(d2h + (uint32_t)((c + 1) * 16), accB);
              act_dot(accA, c);
              ks_tmem_ld_wait();
              if (c + 2 < 4) {
                ks_tmem_ld16(d2h + (uint32_t)((c + 2) * 16), accA);
              } else {                                               // this warpgroup's part of half h is in registers
                ks_tc_fence_before();
                ks_mbar_arrive(bars + BAR_D2_FREE + h);
              }
              act_dot(accB, c + 1);
            }
          }
          z = (z0 + z1) + (z2 + z3);
        }
        // (read after the MMA2 waits: layer 2 of item q is complete, so the producer's t_roof(q) has long been written)
        const float t_roof = ring[(q & (kRing - 1)) * kRows + r];
        // The two column halves meet in shared memory.  Warpgroup 0 (first half of D2, ready one MMA pass
        // earlier) leaves its partial in zpart[q & 1] and moves on; warpgroup 1 picks it up and writes
        // the result.  z_full / z_free hand the two slots back and forth.
        const uint32_t zb = q & 1u, zpar = (q >> 1) & 1u;
        if (wg == 0) {
          if (q >= 2u) ks_mbar_wait(bars + BAR_Z_FREE + zb, zpar ^ 1u);
          zpart[zb * kRows + r] = z;
          ks_mbar_arrive(bars + BAR_Z_FULL + zb);
        } else {
          ks_mbar_wait(bars + BAR_Z_FULL + zb, zpar);
          z += zpart[zb * kRows + r];
          ks_mbar_arrive(bars + BAR_Z_FREE + zb);
        }
        if (wg == 1 && valid) {
          // eta = 1/e, guarded at e >= 2^-10 (Q3): 1 + exp(-z) for one head with a utilisation output,
          // exp(max(z, 0)) with a log-eta output (Q21), k / sum of the members' sigmoids for an
          // ensemble; Eq. 2 floor after eta
          const float eta = fminf(members > 1 ? __fdividef((float)members, z)
                                              : out_add + __expf(fmaxf(out_sgn * (z + b3), out_lo)), 1024.0f);
          lat[(long long)s * bn + row] = fmaxf(t_roof * eta, p.specs.s[s].t0);
        }
      }
    }
  }
}

// ------------------------------------------------------------------ MMA issuer (one elected lane of warp 20)
template <int NIN>
KS_DEV void mma_all(const KsMlpParams& p, const TileMap& tm, const int t_lo, const int t_hi, unsigned char* smem,
                    uint64_t* bars, const uint32_t tmem_base) {
  using C = Cfg256<NIN>;
  constexpr uint32_t idesc = ks_umma_idesc_bf16(128, H);          // layer 1: N = 256
  constexpr uint32_t idesc_half = ks_umma_idesc_bf16(128, H / 2); // layer 2: one column half per pass
  constexpr uint32_t B_LBO = H * 16;
  const uint32_t w1_addr = ks_smem_u32(smem + C::OFF_W1);
  const uint32_t w2_addr = ks_smem_u32(smem + C::OFF_W2);
  const uint32_t a1_addr = ks_smem_u32(smem + C::OFF_A1);
  const uint32_t a2_addr = ks_smem_u32(smem + C::OFF_A2);
  const uint32_t d1 = tmem_base, d2 = tmem_base + (uint32_t)H;
  uint32_t wphase = 0, dphase = 0, q = 0;

  auto mma1 = [&](uint32_t i) {                     // D1 = A1 . W1
    ks_mbar_wait_backoff(bars + BAR_A1_FULL, i & 1u);
    ks_tc_fence_after();
#pragma unroll
    for (int k = 0; k < C::K1 / 16; ++k) {
      const uint64_t ad = ks_umma_desc(a1_addr + k * 2 * kChunkBytes, kChunkBytes, 128);
      const uint64_t bd = ks_umma_desc(w1_addr + k * 2 * B_LBO, B_LBO, 128);
      ks_umma_bf16(d1, ad, bd, idesc, k > 0 ? 1u : 0u);
    }
    ks_umma_commit(bars + BAR_MMA1);
  };
  // Layer 2 runs as two passes over K, one per 128-column half of D2 (W2 rows [128 h, 128 h + 128) =
  // byte offset 2048 h inside every 8-deep K chunk of the image): EPI2's warpgroup 0 activates half 0
  // while the tensor core is still accumulating half 1, and half h of item q+1 only waits for
  // warpgroup h to have drained half h of item q.  With one N = 256 pass the activation of D2 and the
  // next MMA2 could never overlap (D1 + D2 fill TMEM, so D2 cannot be double-buffered).
  auto mma2_group = [&](uint32_t i, int h, int g, bool first, bool last) {   // K group g of D2[half h] += A2 . W2
    if (h == 0) ks_mbar_wait_backoff(bars + BAR_A2_FULL + g, i & 1u);
    if (first && i >= 1u) ks_mbar_wait_backoff(bars + BAR_D2_FREE + h, (i - 1u) & 1u);
    ks_tc_fence_after();
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) {
      const int k16 = g * 4 + kk;
      const uint64_t ad = ks_umma_desc(a2_addr + k16 * 2 * kChunkBytes, kChunkBytes, 128);
      const uint64_t bd = ks_umma_desc(w2_addr + k16 * 2 * B_LBO + h * (H / 2) * 16, B_LBO, 128);
      ks_umma_bf16(d2 + (uint32_t)(h * (H / 2)), ad, bd, idesc_half, (first && kk == 0) ? 0u : 1u);
    }
    if (h == 1) ks_umma_commit(bars + BAR_A2_FREE + g);   // both passes have read this K group: EPI1 may rewrite it
    if (last) {
      if (C::BIAS_MMA) {
        // + b2: whatever item A1 holds by now, its columns 22, 23 are 1 and 24..31 are 0; the features beside them
        // meet zero rows of the bias chunk (finite values: the producers may be rewriting them meanwhile)
        const uint64_t ad = ks_umma_desc(a1_addr + 2 * kChunkBytes, kChunkBytes, 128);   // A1 chunks 2, 3
        const uint64_t bd = ks_umma_desc(ks_smem_u32(smem + C::OFF_B2IMG) + h * (H / 2) * 16, B_LBO, 128);
        ks_umma_bf16(d2 + (uint32_t)(h * (H / 2)), ad, bd, idesc_half, 1u);
      }
      ks_umma_commit(bars + BAR_MMA2 + h);
    }
  };

  for (int b = 0; b < p.n_buckets; ++b) {
    const Range tr = bucket_range(tm, b, t_lo, t_hi);
    if (tr.lo >= tr.hi) continue;
    if (q > 0u) {                                   // every MMA that reads the previous family's weights is done
      ks_umma_commit(bars + BAR_DRAIN);
      ks_mbar_wait_backoff(bars + BAR_DRAIN, dphase);
      dphase ^= 1u;
    }
    ks_mbar_expect_tx(bars + BAR_W, (uint32_t)(C::W1_BYTES + C::W2_BYTES + C::B2IMG_BYTES));
    if (C::BIAS_MMA)
      ks_bulk_g2s(smem + C::OFF_B2IMG, reinterpret_cast<const char*>(p.head[b].w2_img) + (H + 16) * H * 2, C::B2IMG_BYTES,
                  bars + BAR_W);
    ks_bulk_g2s(smem + C::OFF_W1, p.head[b].w1_img, C::W1_BYTES, bars + BAR_W);
    for (int off = 0; off < C::W2_BYTES; off += 32768)
      ks_bulk_g2s(smem + C::OFF_W2 + off, reinterpret_cast<const char*>(p.head[b].w2_img) + off, 32768, bars + BAR_W);
    ks_mbar_wait_backoff(bars + BAR_W, wphase);
    wphase ^= 1u;
    const uint32_t q1 = q + (uint32_t)(tr.hi - tr.lo) * (uint32_t)p.n_specs;
    mma1(q);                                        // D1 is free: the previous family's last item was drained
    for (; q < q1; ++q) {
      mma2_group(q, 0, 0, true, false);
      mma2_group(q, 0, 2, false, false);
      if (q + 1u < q1) {                            // layer 1 of the next item as soon as D1 is drained
        ks_mbar_wait_backoff(bars + BAR_D1_FREE, q & 1u);
        mma1(q + 1u);
      }
      mma2_group(q, 0, 1, false, false);
      mma2_group(q, 0, 3, false, true);
      mma2_group(q, 1, 0, true, false);
      mma2_group(q, 1, 2, false, false);
      mma2_group(q, 1, 1, false, false);
      mma2_group(q, 1, 3, false, true);
    }
  }
}

template <int NIN>
__global__ void __launch_bounds__(kThreads, 1)
ks_mlp_ws256_kernel(const __grid_constant__ KsMlpParams p) {
  using C = Cfg256<NIN>;
  extern __shared__ __align__(1024) unsigned char smem[];
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + BAR_COUNT);
  TileMap* tmp = reinterpret_cast<TileMap*>(smem + C::OFF_BAR + 192);
  const int tid = threadIdx.x;
  const int warp = tid >> 5;

  ks_launch_dependents();     // the step kernel's launch overlaps this kernel (it waits for our completion itself) ...
  cudaGridDependencySynchronize();   // ... as we wait for the kernel before us (ks_launch_pdl)
  if (tid == 32) tile_map_init(p, tmp);
  if (tid == 0) {
    ks_mbar_init(bars + BAR_W, 1);
    ks_mbar_init(bars + BAR_DRAIN, 1);
    ks_mbar_init(bars + BAR_A1_FULL, 128);
    ks_mbar_init(bars + BAR_MMA1, 1);
    ks_mbar_init(bars + BAR_D1_FREE, 256);
    for (int h = 0; h < 2; ++h) {
      ks_mbar_init(bars + BAR_MMA2 + h, 1);
      ks_mbar_init(bars + BAR_D2_FREE + h, p.any_ens ? 128 : 256);   // drained by one warpgroup (ensembles) or by both
      ks_mbar_init(bars + BAR_Z_FULL + h, 128);
      ks_mbar_init(bars + BAR_Z_FREE + h, 128);
    }
    for (int g = 0; g < kGroups; ++g) {
      ks_mbar_init(bars + BAR_A2_FULL + g, 128);
      ks_mbar_init(bars + BAR_A2_FREE + g, 1);
    }
    ks_fence_mbar_init();
  }
  if (warp == 0) { ks_tmem_alloc(tmem_slot, 512); ks_tmem_relinquish(); }
  ks_tc_fence_before();
  __syncthreads();
  ks_tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  const TileMap& tm = *tmp;

  const long long total = tm.tb[p.n_buckets];
  const int t_lo = (int)((long long)blockIdx.x * total / gridDim.x);
  const int t_hi = (int)((long long)(blockIdx.x + 1) * total / gridDim.x);

  if (warp < kProducerWarps) {
    uint32_t q = 0;
    for (int b = 0; b < p.n_buckets; ++b) {
      const Range tr = bucket_range(tm, b, t_lo, t_hi);
      if (tr.lo >= tr.hi) continue;
      switch (p.bk[b].family) {
        case KS_FAM_GEMM: producer_bucket<NIN, KS_FAM_GEMM>(p, tm, b, tr, smem, bars, q); break;
        case KS_FAM_GROUPED_GEMM: producer_bucket<NIN, KS_FAM_GROUPED_GEMM>(p, tm, b, tr, smem, bars, q); break;
        case KS_FAM_ATTN: producer_bucket<NIN, KS_FAM_ATTN>(p, tm, b, tr, smem, bars, q); break;
        default: producer_bucket<NIN, KS_FAM_ELEMWISE>(p, tm, b, tr, smem, bars, q); break;
      }
    }
  } else if (warp < kProducerWarps + kEpiWarps) {
    const uint32_t n_items = (uint32_t)(t_hi - t_lo) * (uint32_t)p.n_specs;
    if (p.gelu_mode == 0) epi1_items<NIN, 0>(p, n_items, smem, bars, tmem_base);
    else epi1_items<NIN, 1>(p, n_items, smem, bars, tmem_base);
  } else if (warp < kMmaWarp) {
    if (p.any_ens) {
      if (p.gelu_mode == 0) epi2_all<NIN, 0, true>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
      else epi2_all<NIN, 1, true>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
    } else {
      if (p.gelu_mode == 0) epi2_all<NIN, 0, false>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
      else epi2_all<NIN, 1, false>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
    }
  } else if (__shfl_sync(0xffffffffu, warp, 0) == kMmaWarp) {   // warp-uniform branch, then one elected lane
    if (ks_elect_one()) mma_all<NIN>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
  }
  ks_tc_fence_before();
  __syncthreads();
  if (warp == 0) ks_tmem_dealloc(tmem_base, 512);
}

template <int NIN>
cudaError_t launch_ws256(const KsMlpParams& p, int num_sms, cudaStream_t st) {
  using C = Cfg256<NIN>;
  const int total = p.tile_begin[p.n_buckets];
  if (total <= 0) return cudaSuccess;
  const int grid = total < num_sms ? total : num_sms;
  auto kern = ks_mlp_ws256_kernel<NIN>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  return ks_launch_pdl(kern, grid, kThreads, C::SMEM_BYTES, st, p);
}

}  // namespace

cudaError_t ks_launch_mlp_ws256(const KsMlpParams& p, int n_in, int num_sms, cudaStream_t st) {
  if (n_in == 8) return launch_ws256<8>(p, num_sms, st);
  if (n_in == 12) return launch_ws256<12>(p, num_sms, st);
  if (n_in == 32) return launch_ws256<32>(p, num_sms, st);
  return cudaErrorInvalidValue;
}
