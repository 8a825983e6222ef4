// ks_mlp_pool256.cu — Tier-A kernel for H = 256 (cfg5) with a POOL of six activation warpgroups.
// S1-S3, S4a, S5 of DESIGN.md §1 (PAPER.md:191 Eq. 2, :199-201 per-family heads), fused; same producers, same MMA
// issuer, same shared-memory and TMEM layout as ks_mlp_ws256.cu.  What differs is who activates what.
//
// A clock64 trace of ks_mlp_ws256.cu (profiles/README.md) shows its four activation warpgroups busy 93 % of the time
// while the MUFU pipe is 68 % and the issue port 53 % busy: with five warps per SM sub-partition and ~6 instructions
// around every MUFU.TANH the warps cannot hide one another's latencies.  Here an item's activation work is cut into EIGHT
// uniform units of 64 columns -- units 0-3: D1 columns [64 k, 64 k + 64) -> A2 K group k (layer 1's GELU); units 4-7:
// D2 half h, columns [128 h + 64 part, + 64) (layer 2's GELU and the dot with w3) -- and unit u of item q goes to
// warpgroup (8 q + u) mod 6 of SIX warpgroups (24 warps: seven warps per sub-partition with the producers).  Every
// dependency of a unit is a unit with a smaller sequence number 8 q + u (through an mbarrier or through the tensor
// core) and a warpgroup takes its units in increasing order, so the pipeline cannot deadlock; both kinds of unit are in
// flight at once (layer 1 of item q+1 beside layer 2 of item q) whatever their relative cost.
// The four partial dot products of an item meet in shared memory: units 4-6 leave theirs in a two-slot buffer
// (z_full / z_free), unit 7 adds them in a fixed order and writes the latency.  Per-family w3 / b2 are staged by the
// issuer's TMA together with the weights, double-buffered by family.  Ensembles stay on ks_mlp_ws256.cu.
#include <type_traits>
#include "ks_mlp_common.cuh"
#ifndef KS_POOL_SETMAXNREG
#define KS_POOL_SETMAXNREG 0
#endif

namespace {

using namespace ksmlp;

constexpr int H = 256;
constexpr int kProducerWarps = 4, kPoolGroups = 6, kPoolWarps = 4 * kPoolGroups;
constexpr int kMmaWarp = kProducerWarps + kPoolWarps;               // warp 28
constexpr int kThreads = 1024;                                      // eight whole warpgroups (warps 29-31 idle)
constexpr int kRing = 4;
constexpr int kGroups = 4;                                          // A2 K groups of 64 columns
// registers per thread after the roles have re-divided the CTA's allocation (setmaxnreg; 1024 x 64 at launch)
constexpr int kRegsProducer = 56, kRegsPool = 72, kRegsMma = 24;
static_assert(128 * kRegsProducer + 768 * kRegsPool + 128 * kRegsMma <= 65536, "register budget");

template <int NIN>
struct Cfg256 {
  static constexpr int K1 = NIN == 32 ? 32 : 16;
  static constexpr int BIAS_ROW = NIN == 32 ? 22 : NIN;
  static constexpr int W1_BYTES = K1 * H * 2;
  static constexpr int W2_BYTES = H * H * 2;       // K rows 0..H-1 of the image: the bias rows are not staged
  static constexpr int A1_BYTES = (K1 / 8) * kChunkBytes;
  static constexpr int A2_BYTES = (H / 8) * kChunkBytes;
  static constexpr int OFF_W1 = 0;
  static constexpr int OFF_W2 = OFF_W1 + W1_BYTES;
  static constexpr int OFF_A1 = OFF_W2 + W2_BYTES;
  static constexpr int OFF_A2 = OFF_A1 + A1_BYTES;
  static constexpr int OFF_W3 = OFF_A2 + A2_BYTES;            // [2][H] fp32 w3/2, by family parity
  static constexpr int OFF_B2 = OFF_W3 + 2 * H * 4;           // [2][H] fp32 b2
  static constexpr int OFF_RING = OFF_B2 + 2 * H * 4;         // [kRing][128] fp32 t_roof
  static constexpr int OFF_ZP = OFF_RING + kRing * kRows * 4; // [2][3][128] fp32 partial dots of units 4-6
  static constexpr int OFF_BAR = OFF_ZP + 2 * 3 * kRows * 4;
  static constexpr int SMEM_BYTES = OFF_BAR + 320;   // 21 barriers, TMEM slot (240), TileMap (256)
};

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

// ------------------------------------------------------------------ the activation pool (warps 4-27)
template <int NIN, int GM>
KS_DEV void pool_units(const KsMlpParams& p, const TileMap& tm, const int t_lo, const int t_hi, unsigned char* smem,
                       uint64_t* bars, const uint32_t tmem_base) {
  using C = Cfg256<NIN>;
  const int e = threadIdx.x - kProducerWarps * 32;                  // 0..767
  const uint32_t g = (uint32_t)e >> 7;                              // warpgroup 0..5
  const int r = e & 127;
  const uint32_t lane_off = (uint32_t)((r >> 5) * 32) << 16;
  unsigned char* A2 = smem + C::OFF_A2;
  const float* ring = reinterpret_cast<const float*>(smem + C::OFF_RING);
  const float* sw3_all = reinterpret_cast<const float*>(smem + C::OFF_W3);
  const float* sb2_all = reinterpret_cast<const float*>(smem + C::OFF_B2);
  float* zpart = reinterpret_cast<float*>(smem + C::OFF_ZP);
  const uint32_t n_specs = (uint32_t)p.n_specs;
  const uint32_t n_units = (uint32_t)(t_hi - t_lo) * n_specs * 8u;
#pragma unroll 1
  for (uint32_t sq = g; sq < n_units; sq += (uint32_t)kPoolGroups) {
    const uint32_t q = sq >> 3, par = q & 1u;
    const int u = (int)(sq & 7u);
    uint32_t accA[16], accB[16];
    if (u < 4) {
      // ---- layer 1: D1 columns [64 u, 64 u + 64) -> 2 GELU -> bf16 -> A2 K group u
      ks_mbar_wait(bars + BAR_MMA1, par);                           // D1 holds item q
      ks_tc_fence_after();
      const uint32_t d1 = tmem_base + lane_off + (uint32_t)(u * 64);
      ks_tmem_ld16(d1, accA);
      auto act_store = [&](const uint32_t* a, int c16, bool wait_free) {
        uint32_t pk[8];
        if (GM == 0) {
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            float g0, g1;
            gelu2_f32x2(__uint_as_float(a[2 * j]), __uint_as_float(a[2 * j + 1]), g0, g1);
            pk[j] = ks_pack_bf16x2_alu(g0, g1);
          }
        } else {
#pragma unroll
          for (int j = 0; j < 8; ++j) pk[j] = gelu2_bf16x2(__uint_as_float(a[2 * j]), __uint_as_float(a[2 * j + 1]));
        }
        // the group is stored once MMA2(q-1) has read it (both passes); the wait sits behind the first arithmetic
        if (wait_free) ks_mbar_wait(bars + BAR_A2_FREE + u, par ^ 1u);
        const int kc = u * 8 + c16 * 2;                             // 8-column K chunk index
        *reinterpret_cast<uint4*>(A2 + (kc + 0) * kChunkBytes + r * 16) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
        *reinterpret_cast<uint4*>(A2 + (kc + 1) * kChunkBytes + r * 16) = make_uint4(pk[4], pk[5], pk[6], pk[7]);
      };
#pragma unroll 1
      for (int c = 0; c < 4; c += 2) {
        ks_tmem_ld_wait();
        ks_tmem_ld16(d1 + (uint32_t)((c + 1) * 16), accB);
        act_store(accA, c, c == 0 && q >= 1u);
        ks_tmem_ld_wait();
        if (c + 2 < 4) {
          ks_tmem_ld16(d1 + (uint32_t)((c + 2) * 16), accA);
        } else {                                                    // this unit's part of D1 is in registers
          ks_tc_fence_before();
          ks_mbar_arrive(bars + BAR_D1_FREE);
        }
        act_store(accB, c + 1, false);
      }
      ks_fence_proxy_async();
      ks_mbar_arrive(bars + BAR_A2_FULL + u);
    } else {
      // ---- layer 2: D2 half h, columns [128 h + 64 part, + 64): + b2 -> 2 GELU -> dot with w3/2
      const int h = (u - 4) >> 1, part = (u - 4) & 1;
      // the family of item q (tile t) and its parity among the families this CTA meets (the issuer stages w3 / b2 by it)
      const int t = t_lo + (int)(q / n_specs);
      int b = 0, bseq = 0;
      for (int bb = 0; bb + 1 < p.n_buckets; ++bb)
        if (t >= tm.tb[bb + 1]) { b = bb + 1; }
      for (int bb = 0; bb < b; ++bb) {
        const Range tr = bucket_range(tm, bb, t_lo, t_hi);
        bseq += tr.lo < tr.hi ? 1 : 0;
      }
      const float* sw3 = sw3_all + (bseq & 1) * H;
      const float* sb2 = sb2_all + (bseq & 1) * H;
      ks_mbar_wait(bars + BAR_MMA2 + h, par);                       // half h of D2 holds item q
      ks_tc_fence_after();
      const int col0 = h * 128 + part * 64;
      const uint32_t d2h = tmem_base + (uint32_t)H + lane_off + (uint32_t)col0;
      ks_tmem_ld16(d2h, accA);
      float z0 = 0.0f, z1 = 0.0f, z2 = 0.0f, z3 = 0.0f;
      auto act_dot = [&](const uint32_t* a, int c16) {
        const int col = col0 + c16 * 16;
#pragma unroll
        for (int j = 0; j < 16; j += 4) {
          const float4 w4 = *reinterpret_cast<const float4*>(sw3 + col + j);
          const float4 b4 = *reinterpret_cast<const float4*>(sb2 + col + j);
          float x0, x1, x2, x3;
          ks_add2(x0, x1, __uint_as_float(a[j + 0]), __uint_as_float(a[j + 1]), b4.x, b4.y);
          ks_add2(x2, x3, __uint_as_float(a[j + 2]), __uint_as_float(a[j + 3]), b4.z, b4.w);
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
        } else {                                                    // this unit's part of half h is in registers
          ks_tc_fence_before();
          ks_mbar_arrive(bars + BAR_D2_FREE + h);
        }
        act_dot(accB, c + 1);
      }
      float z = (z0 + z1) + (z2 + z3);
      const uint32_t zb = q & 1u, zpar = (q >> 1) & 1u;
      if (u != 7) {
        if (q >= 2u) ks_mbar_wait(bars + BAR_Z_FREE + zb, zpar ^ 1u);   // unit 7 of item q-2 has read the slot
        zpart[(zb * 3 + (uint32_t)(u - 4)) * kRows + r] = z;
        ks_mbar_arrive(bars + BAR_Z_FULL + zb);
      } else {
        ks_mbar_wait(bars + BAR_Z_FULL + zb, zpar);
        z = ((zpart[(zb * 3 + 0) * kRows + r] + zpart[(zb * 3 + 1) * kRows + r]) + zpart[(zb * 3 + 2) * kRows + r]) + z;
        ks_mbar_arrive(bars + BAR_Z_FREE + zb);
        const float t_roof = ring[(q & (kRing - 1)) * kRows + r];
        const KsBucketDev& bk = p.bk[b];
        const KsHeadDev& hd = p.head[b];
        const int pos = (t - tm.tb[b]) * kRows + r;
        if (pos < tm.ne[b]) {
          const int row = bk.idx ? __ldg(bk.idx + pos) : pos;
          const uint32_t s = q - (q / n_specs) * n_specs;
          // eta = 1/e, guarded at e >= 2^-10 (Q3): 1 + exp(-z) with a utilisation output, exp(max(z, 0)) with a
          // log-eta output (Q21); Eq. 2 floor after eta
          const float eta = fminf(hd.out_add + __expf(fmaxf(hd.out_sgn * (z + hd.b3), hd.out_lo)), 1024.0f);
          bk.lat[(long long)s * bk.n + row] = fmaxf(t_roof * eta, p.specs.s[s].t0);
        }
      }
    }
  }
}

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
    if (last) ks_umma_commit(bars + BAR_MMA2 + h);
  };

  for (int b = 0; b < p.n_buckets; ++b) {
    const Range tr = bucket_range(tm, b, t_lo, t_hi);
    if (tr.lo >= tr.hi) continue;
    if (q > 0u) {                                   // every MMA that reads the previous family's weights is done
      ks_umma_commit(bars + BAR_DRAIN);
      ks_mbar_wait_backoff(bars + BAR_DRAIN, dphase);
      dphase ^= 1u;
    }
    ks_mbar_expect_tx(bars + BAR_W, (uint32_t)(C::W1_BYTES + C::W2_BYTES + 2 * H * 4));
    ks_bulk_g2s(smem + C::OFF_W3 + (int)wphase * H * 4, p.head[b].w3, H * 4, bars + BAR_W);   // by family parity
    ks_bulk_g2s(smem + C::OFF_B2 + (int)wphase * H * 4, p.head[b].b2, H * 4, bars + BAR_W);
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
ks_mlp_pool256_kernel(const __grid_constant__ KsMlpParams p) {
  using C = Cfg256<NIN>;
  extern __shared__ __align__(1024) unsigned char smem[];
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + C::OFF_BAR + 240);
  TileMap* tmp = reinterpret_cast<TileMap*>(smem + C::OFF_BAR + 256);
  static_assert(BAR_COUNT * 8 <= 240 && sizeof(TileMap) <= 64, "barrier block layout");
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
    ks_mbar_init(bars + BAR_D1_FREE, 512);          // four units of 128 threads
    for (int h = 0; h < 2; ++h) {
      ks_mbar_init(bars + BAR_MMA2 + h, 1);
      ks_mbar_init(bars + BAR_D2_FREE + h, 256);    // two units
      ks_mbar_init(bars + BAR_Z_FULL + h, 384);     // units 4-6
      ks_mbar_init(bars + BAR_Z_FREE + h, 128);     // unit 7
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
#if KS_POOL_SETMAXNREG
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsProducer));
#endif
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
  } else if (warp < kMmaWarp) {
#if KS_POOL_SETMAXNREG
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsPool));
#endif
    if (p.gelu_mode == 0) pool_units<NIN, 0>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
    else pool_units<NIN, 1>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
  } else {                                                      // warps 28-31: the issuer's warpgroup
#if KS_POOL_SETMAXNREG
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsMma));
#endif
    if (__shfl_sync(0xffffffffu, warp, 0) == kMmaWarp) {        // warp-uniform branch, then one elected lane
      if (ks_elect_one()) mma_all<NIN>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
    }
  }
  ks_tc_fence_before();
  __syncthreads();
  if (warp == 0) ks_tmem_dealloc(tmem_base, 512);
}

template <int NIN>
cudaError_t launch_pool256(const KsMlpParams& p, int num_sms, cudaStream_t st) {
  using C = Cfg256<NIN>;
  const int total = p.tile_begin[p.n_buckets];
  if (total <= 0) return cudaSuccess;
  const int grid = total < num_sms ? total : num_sms;
  auto kern = ks_mlp_pool256_kernel<NIN>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  return ks_launch_pdl(kern, grid, kThreads, C::SMEM_BYTES, st, p);
}

}  // namespace

cudaError_t ks_launch_mlp_pool256(const KsMlpParams& p, int n_in, int num_sms, cudaStream_t st) {
  if (n_in == 8) return launch_pool256<8>(p, num_sms, st);
  if (n_in == 12) return launch_pool256<12>(p, num_sms, st);
  if (n_in == 32) return launch_pool256<32>(p, num_sms, st);
  return cudaErrorInvalidValue;
}
