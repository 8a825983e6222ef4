// ks_mlp_ws.cu — Tier-A kernel for H <= 128: a warp-specialized pipeline around the 5th-gen tensor
// cores.  S1-S3, S4a, S5 of DESIGN.md §1 (PAPER.md:191 Eq. 2, :199-201 per-family heads), fused.
//
// One persistent CTA per SM walks a contiguous range of 128-row tiles.  A work item q is one
// (tile, spec) pair; item q uses buffer q & 1 of every double-buffered resource (A1, D1, D2) and
// buffer q % 3 of the layer-2 operand A2.
//
//   warps 0-3    PRODUCER  thread r owns row r: prefetch next tile's columns, decode + roofline +
//                          features -> bf16 A1[q&1] row in smem (K-major UMMA image), t_roof -> ring
//   warp  20     MMA       one thread: MMA1(q+2): D1 = A1 . W1 (b1 rides on two 1-columns) as soon as
//                          EPI1 has drained D1[q&1]; then MMA2(q): D2 = A2 . W2 (+ ones-block x b2 step)
//   warps 4-11   EPI1      two warpgroups, group g owns buffer g: D1 -> regs (tcgen05.ld, 16 columns,
//                          double-buffered) -> 2 GELU -> bf16 -> A2[g] in smem
//   warps 12-19  EPI2      same split: D2 -> regs -> 2 GELU -> fp32 dot with w3/2 -> sigmoid -> latency
//
// so the tensor core, the activation warps of layer 1 and of layer 2 and the feature warps all work
// on different items at the same time; nobody waits for its own MMA.  Synchronisation is by
// mbarriers only (no CTA-wide barrier in the loop):
//   a1_full[2]   128 producer arrivals      -> MMA may read A1[b]
//   mma1_done[2] tcgen05.commit             -> EPI1 may read D1[b]; producer may rewrite A1[b]
//   d1_free[2]   128 EPI1 arrivals          -> D1[b] has been drained: MMA1(q+2) may overwrite it
//   a2_full[3]   128 EPI1 arrivals          -> MMA may read A2[q % 3]
//   mma2_done[2] tcgen05.commit             -> EPI2 may read D2[b]
//   a2_free[3]   tcgen05.commit             -> MMA2(q) has read A2[q % 3]: EPI1 of item q + 3 may rewrite it
//   d2_free[2]   128 EPI2 arrivals          -> D2[b] has been drained: MMA2(q+2) may overwrite it
// A2 has three buffers and D1/D2 are released as soon as their last tcgen05.ld has completed, because
// the warpgroup that finishes item q is the one that continues with item q + 2 of the same buffer: with
// two A2 buffers (or a late release) it would sit out a whole MMA2 per item (cycle trace of one CTA:
// ~1100 of ~6300 cycles per item and group).
// A waiter for completion k of a barrier always runs before completion k+1 can happen (k+1 depends
// on the waiter's own progress), so single-bit phase parity is sufficient.
// The t_roof ring has 8 entries: the producer can be at most 7 items ahead of EPI2 (item q+8 needs
// mma1_done(q+6); MMA1(q+6) is issued after MMA2(q+3), which waits for d2_free(q+1) >= d2_free(q)).
#include <type_traits>
#include "ks_mlp_common.cuh"

namespace {

using namespace ksmlp;

// Each epilogue role has two warpgroups: group g takes the items with q & 1 == g, i.e. it owns
// buffer g.  Four activation warps per SM sub-partition keep the MUFU pipe fed while any one of
// them waits for its next accumulator.
constexpr int kProducerWarps = 4, kEpiWarps = 8;
constexpr int kWsThreads = (kProducerWarps + 2 * kEpiWarps + 1) * 32;   // 672
constexpr int kMmaWarp = kProducerWarps + 2 * kEpiWarps;
constexpr int kRing = 8;
constexpr int kA2Bufs = 3;     // A2 (layer-2 operand) is triple-buffered: item q uses A2[q % 3]

template <int NIN, int H>
struct WsCfg {
  static constexpr int K1 = NIN == 32 ? 32 : 16;
  static constexpr int BIAS_ROW = NIN == 32 ? 22 : NIN;
  static constexpr int TMEM_COLS = 4 * H;              // D1[2], D2[2]
  static constexpr int W1_BYTES = K1 * H * 2;
  static constexpr int W2_BYTES = (H + 16) * H * 2;
  static constexpr int A1_BYTES = (K1 / 8) * kChunkBytes;
  static constexpr int A2_BYTES = (H / 8) * kChunkBytes;
  static constexpr int ONES_BYTES = 2 * kChunkBytes;
  static constexpr int OFF_W1 = 0;
  static constexpr int OFF_W2 = OFF_W1 + W1_BYTES;
  static constexpr int OFF_ONES = OFF_W2 + W2_BYTES;
  static constexpr int OFF_A1 = OFF_ONES + ONES_BYTES;
  static constexpr int OFF_A2 = OFF_A1 + 2 * A1_BYTES;
  static constexpr int OFF_W3 = OFF_A2 + kA2Bufs * A2_BYTES;           // [KS_MLP_MAX_BUCKETS][H] fp32
  static constexpr int OFF_RING = OFF_W3 + KS_MLP_MAX_BUCKETS * H * 4; // [kRing][128] fp32 t_roof
  static constexpr int OFF_BAR = OFF_RING + kRing * kRows * 4;
  static constexpr int SMEM_BYTES = OFF_BAR + 224;   // barriers + TMEM slot (160) + TileMap
};

// barrier slots inside the OFF_BAR block
enum { BAR_W = 0, BAR_DRAIN = 1, BAR_A1_FULL = 2, BAR_MMA1 = 4, BAR_A2_FULL = 6, BAR_MMA2 = 9, BAR_D2_FREE = 11,
       BAR_D1_FREE = 13, BAR_A2_FREE = 15, BAR_COUNT = 18 };

struct Range { int lo, hi; };
KS_DEV Range bucket_range(const TileMap& tm, int b, int t_lo, int t_hi) {
  Range r;
  r.lo = t_lo > tm.tb[b] ? t_lo : tm.tb[b];
  r.hi = t_hi < tm.tb[b + 1] ? t_hi : tm.tb[b + 1];
  return r;
}

// ------------------------------------------------------------------ PRODUCER (warps 0-3)
template <int NIN, int H, int FAM>
KS_DEV void producer_bucket(const KsMlpParams& p, const TileMap& tm, const int b, const Range tr, unsigned char* smem,
                            uint64_t* bars, uint32_t& q) {
  using C = WsCfg<NIN, H>;
  constexpr int NC = NCols<FAM>::v;
  const int r = threadIdx.x;                       // 0..127: row within the tile
  const KsBucketDev& bk = p.bk[b];
  const int tile0 = tm.tb[b], ne = tm.ne[b];
  const bool f32cols = bk.col_f32 != 0;
  float* ring = reinterpret_cast<float*>(smem + C::OFF_RING);

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
      const uint32_t buf = q & 1u;
      if (q >= 2u) ks_mbar_wait(bars + BAR_MMA1 + buf, ((q >> 1) - 1u) & 1u);   // MMA1(q-2) has consumed A1[buf]
      unsigned char* A1 = smem + C::OFF_A1 + buf * C::A1_BYTES;
#pragma unroll
      for (int kc = 0; kc < C::K1 / 8; ++kc) *reinterpret_cast<uint4*>(A1 + kc * kChunkBytes + r * 16) = a1[kc];
      ring[(q & (kRing - 1)) * kRows + r] = t_roof;
      ks_fence_proxy_async();                      // generic-proxy stores -> visible to the tensor core
      ks_mbar_arrive(bars + BAR_A1_FULL + buf);
    }
  }
}

// ------------------------------------------------------------------ EPI1 (warps 4-11): D1 -> 2 GELU -> A2
template <int NIN, int H, int GM>
KS_DEV void epi1_items(const KsMlpParams& p, const uint32_t n_items, unsigned char* smem, uint64_t* bars,
                       const uint32_t tmem_base) {
  using C = WsCfg<NIN, H>;
  const int e = threadIdx.x - kProducerWarps * 32;
  const uint32_t grp = (uint32_t)e >> 7;                           // warpgroup of this role: owns buffer grp
  const int r = e & 127;                                           // TMEM lane = tile row
  const uint32_t lane_off = (uint32_t)((r >> 5) * 32) << 16;
  uint32_t a2i = grp, a2p = 0;                                     // q % 3 and the parity of q / 3
  for (uint32_t q = grp; q < n_items; q += 2) {
    const uint32_t buf = q & 1u, par = (q >> 1) & 1u;
    unsigned char* A2 = smem + C::OFF_A2 + a2i * C::A2_BYTES;
    const uint32_t d1 = tmem_base + buf * H + lane_off;
    ks_mbar_wait(bars + BAR_MMA1 + buf, par);                       // D1[buf] holds item q
    ks_tc_fence_after();
    // 16-column sub-chunks, double-buffered in registers: the load of sub-chunk c+1 is in flight
    // while c is activated.  The loop stays rolled (two sub-chunks per trip) so the code of all
    // roles together fits the 32 KB instruction cache.
    uint32_t accA[16], accB[16];
    ks_tmem_ld16(d1, accA);
    // MMA2(q-3) has consumed A2[q % 3].  With two A2 buffers this group would sit out the whole MMA2(q-2),
    // which can only start when the group's previous item is finished (measured: ~1100 of ~6300 cycles).
    if (q >= 3u) ks_mbar_wait(bars + BAR_A2_FREE + a2i, a2p ^ 1u);
    auto act_store = [&](const uint32_t* a, int c16) {
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
      *reinterpret_cast<uint4*>(A2 + (c16 * 2 + 0) * kChunkBytes + r * 16) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
      *reinterpret_cast<uint4*>(A2 + (c16 * 2 + 1) * kChunkBytes + r * 16) = make_uint4(pk[4], pk[5], pk[6], pk[7]);
    };
#pragma unroll 1
    for (int c = 0; c < H / 16; c += 2) {
      ks_tmem_ld_wait();
      ks_tmem_ld16(d1 + (uint32_t)((c + 1) * 16), accB);
      act_store(accA, c);
      ks_tmem_ld_wait();
      if (c + 2 < H / 16) {
        ks_tmem_ld16(d1 + (uint32_t)((c + 2) * 16), accA);
      } else {                                     // D1[buf] is drained: MMA1(q+2) may overwrite it now
        ks_tc_fence_before();
        ks_mbar_arrive(bars + BAR_D1_FREE + buf);
      }
      act_store(accB, c + 1);
    }
    ks_fence_proxy_async();
    ks_mbar_arrive(bars + BAR_A2_FULL + a2i);
    a2i += 2u;
    if (a2i >= 3u) { a2i -= 3u; a2p ^= 1u; }
  }
}

// ------------------------------------------------------------------ EPI2 (warps 12-19): D2 -> 2 GELU . w3/2 -> latency
template <int NIN, int H, int GM, bool ENS>
KS_DEV void epi2_all(const KsMlpParams& p, const TileMap& tm, const int t_lo, const int t_hi, unsigned char* smem,
                     uint64_t* bars, const uint32_t tmem_base) {
  using C = WsCfg<NIN, H>;
  const int e = threadIdx.x - (kProducerWarps + kEpiWarps) * 32;
  const uint32_t grp = (uint32_t)e >> 7;
  const int r = e & 127;
  const uint32_t lane_off = (uint32_t)((r >> 5) * 32) << 16;
  const float* ring = reinterpret_cast<const float*>(smem + C::OFF_RING);
  uint32_t q = 0;
  for (int b = 0; b < p.n_buckets; ++b) {
    const Range tr = bucket_range(tm, b, t_lo, t_hi);
    const KsBucketDev& bk = p.bk[b];
    const float* sw3 = reinterpret_cast<const float*>(smem + C::OFF_W3) + b * H;
    const KsHeadDev& hd = p.head[b];
    const float b3 = hd.b3, out_sgn = hd.out_sgn, out_lo = hd.out_lo, out_add = hd.out_add;
    const int members = ENS ? hd.members : 1;                                  // > 1: MLP ensemble, members of H / members columns
    const int ens_mask = members > 1 ? H / 16 / members - 1 : 0;     // member width is 32 or 64: a power-of-two chunk count
    const int tile0 = tm.tb[b], ne = tm.ne[b];
    // Everything the item loop needs from the kernel parameters is read once per bucket into registers
    // (the asm keeps the compiler from re-reading it with indexed constant loads on every item: measured
    // ~900 idle cycles between two items of a group), and a thread only walks its own group's items.
    const int* idx = bk.idx;
    float* lat = bk.lat;
    int bn = bk.n, n_specs = p.n_specs;
    asm volatile("" : "+l"(idx), "+l"(lat), "+r"(bn), "+r"(n_specs));
    const uint32_t n_it = tr.lo < tr.hi ? (uint32_t)(tr.hi - tr.lo) * (uint32_t)n_specs : 0u;
    const uint32_t q0 = q;
    q += n_it;
    int t = tr.lo, s = (int)((q0 & 1u) ^ grp);       // first item of this group in the bucket: i = (q0 & 1) ^ grp
    while (n_it != 0u && s >= n_specs) { s -= n_specs; ++t; }
    for (uint32_t i = (q0 & 1u) ^ grp; i < n_it; i += 2u) {
      const uint32_t qi = q0 + i;
      {
        const int pos = (t - tile0) * kRows + r;
        const bool valid = pos < ne;
        const int row = valid ? (idx ? __ldg(idx + pos) : pos) : 0;
        const uint32_t buf = qi & 1u, par = (qi >> 1) & 1u;
        const uint32_t d2 = tmem_base + 2 * H + buf * H + lane_off;
        ks_mbar_wait(bars + BAR_MMA2 + buf, par);                   // D2[buf] holds item q
        ks_tc_fence_after();
        uint32_t accA[16], accB[16];
        ks_tmem_ld16(d2, accA);
        const float t_roof = ring[(qi & (kRing - 1)) * kRows + r];
        float t0 = p.specs.s[s].t0;                 // (an indexed constant load: issued here, used after the sweep)
        asm volatile("" : "+f"(t0));
        float z0 = 0.0f, z1 = 0.0f, z2 = 0.0f, z3 = 0.0f;
        auto act_dot = [&](const uint32_t* a, int c16) {
          if (GM == 0) {
#pragma unroll
            for (int j = 0; j < 16; j += 4) {
              const float4 w4 = *reinterpret_cast<const float4*>(sw3 + c16 * 16 + j);
              float g0, g1, g2, g3;
              gelu2_f32x2(__uint_as_float(a[j + 0]), __uint_as_float(a[j + 1]), g0, g1);
              gelu2_f32x2(__uint_as_float(a[j + 2]), __uint_as_float(a[j + 3]), g2, g3);
              ks_fma2(z0, z1, g0, g1, w4.x, w4.y, z0, z1);
              ks_fma2(z2, z3, g2, g3, w4.z, w4.w, z2, z3);
            }
          } else {
#pragma unroll
            for (int j = 0; j < 16; j += 4) {
              const float4 w4 = *reinterpret_cast<const float4*>(sw3 + c16 * 16 + j);
              const uint32_t g0 = gelu2_bf16x2(__uint_as_float(a[j + 0]), __uint_as_float(a[j + 1]));
              const uint32_t g1 = gelu2_bf16x2(__uint_as_float(a[j + 2]), __uint_as_float(a[j + 3]));
              z0 = fmaf(__uint_as_float(g0 << 16), w4.x, z0);
              z1 = fmaf(__uint_as_float(g0 & 0xffff0000u), w4.y, z1);
              z2 = fmaf(__uint_as_float(g1 << 16), w4.z, z2);
              z3 = fmaf(__uint_as_float(g1 & 0xffff0000u), w4.w, z3);
            }
          }
        };
        float esum = 0.0f;                         // ensemble: sum of the members' efficiencies so far
        auto sweep = [&](auto ens) {
          int m = 0;
#pragma unroll 1
          for (int c = 0; c < H / 16; c += 2) {
            ks_tmem_ld_wait();
            ks_tmem_ld16(d2 + (uint32_t)((c + 1) * 16), accB);
            act_dot(accA, c);
            ks_tmem_ld_wait();
            if (c + 2 < H / 16) {
              ks_tmem_ld16(d2 + (uint32_t)((c + 2) * 16), accA);
            } else {
              // D2[buf] is drained: MMA2(q+2) may overwrite it while the last sub-chunk is still being
              // activated.  This group is the one that will wait for that MMA2 (measured: a bubble of a
              // whole MMA2, ~1150 cycles per item, when the release came after the loop).
              ks_tc_fence_before();
              ks_mbar_arrive(bars + BAR_D2_FREE + buf);
            }
            act_dot(accB, c + 1);
            if (decltype(ens)::value && ((c + 2) & ens_mask) == 0) {   // last column of member m (Q17)
              const float z = ((z0 + z1) + (z2 + z3)) + hd.b3m[m++];
              esum += __fdividef(1.0f, 1.0f + __expf(-z));
              z0 = z1 = z2 = z3 = 0.0f;
            }
          }
        };
        if (members > 1) sweep(std::true_type{}); else sweep(std::false_type{});
        if (valid) {
          float eta;
          if (members > 1) {
            // e = mean of the members' sigmoids; eta = 1/e with the same guard e >= 2^-10
            eta = fminf(__fdividef((float)members, esum), 1024.0f);
          } else {
            const float z = ((z0 + z1) + (z2 + z3)) + b3;
            // eta = 1/e = 1 + exp(-z) (utilisation output), or exp(max(z, 0)) (log-eta output; Q21);
            // guarded at e >= 2^-10 (Q3); Eq. 2 floor after eta
            eta = fminf(out_add + __expf(fmaxf(out_sgn * z, out_lo)), 1024.0f);
          }
          lat[(long long)s * bn + row] = fmaxf(t_roof * eta, t0);
        }
      }
      s += 2;
      while (s >= n_specs) { s -= n_specs; ++t; }
    }
  }
}

// ------------------------------------------------------------------ MMA issuer (one thread of warp 20)
template <int NIN, int H>
KS_DEV void mma_all(const KsMlpParams& p, const TileMap& tm, const int t_lo, const int t_hi, unsigned char* smem,
                    uint64_t* bars, const uint32_t tmem_base) {
  using C = WsCfg<NIN, H>;
  constexpr uint32_t idesc = ks_umma_idesc_bf16(128, H);
  constexpr uint32_t B_LBO = H * 16;
  const uint32_t w1_addr = ks_smem_u32(smem + C::OFF_W1);
  const uint32_t w2_addr = ks_smem_u32(smem + C::OFF_W2);
  const uint32_t ones_addr = ks_smem_u32(smem + C::OFF_ONES);
  const uint32_t a1_addr = ks_smem_u32(smem + C::OFF_A1);
  const uint32_t a2_addr = ks_smem_u32(smem + C::OFF_A2);
  uint32_t wphase = 0, dphase = 0, q = 0;
  uint32_t m2i = 0, m2p = 0;                        // A2 buffer (q % 3) and parity of q / 3 of the next MMA2

  auto mma2 = [&](uint32_t i) {                     // D2[i&1] = A2[i&1] . W2 + ones x b2
    const uint32_t buf = i & 1u, par = (i >> 1) & 1u;
    ks_mbar_wait_backoff(bars + BAR_A2_FULL + m2i, m2p);
    if (i >= 2u) ks_mbar_wait_backoff(bars + BAR_D2_FREE + buf, par ^ 1u);
    ks_tc_fence_after();
    const uint32_t d2 = tmem_base + 2 * H + buf * H;
    const uint32_t a = a2_addr + m2i * C::A2_BYTES;
#pragma unroll
    for (int k16 = 0; k16 < H / 16; ++k16) {
      const uint64_t ad = ks_umma_desc(a + k16 * 2 * kChunkBytes, kChunkBytes, 128);
      const uint64_t bd = ks_umma_desc(w2_addr + k16 * 2 * B_LBO, B_LBO, 128);
      ks_umma_bf16(d2, ad, bd, idesc, k16 > 0 ? 1u : 0u);
    }
    const uint64_t ad = ks_umma_desc(ones_addr, kChunkBytes, 128);
    const uint64_t bd = ks_umma_desc(w2_addr + (H / 8) * B_LBO, B_LBO, 128);
    ks_umma_bf16(d2, ad, bd, idesc, 1u);
    ks_umma_commit(bars + BAR_MMA2 + buf);          // D2[buf] is complete (EPI2)
    ks_umma_commit(bars + BAR_A2_FREE + m2i);       // ... and A2[q % 3] has been read (EPI1 of item q + 3)
    if (++m2i == 3u) { m2i = 0; m2p ^= 1u; }
  };

  auto mma1 = [&](uint32_t i) {                     // D1[i&1] = A1[i&1] . W1
    const uint32_t buf = i & 1u, par = (i >> 1) & 1u;
    ks_mbar_wait_backoff(bars + BAR_A1_FULL + buf, par);
    ks_tc_fence_after();
    const uint32_t d1 = tmem_base + buf * H;
    const uint32_t a = a1_addr + buf * C::A1_BYTES;
#pragma unroll
    for (int k = 0; k < C::K1 / 16; ++k) {
      const uint64_t ad = ks_umma_desc(a + k * 2 * kChunkBytes, kChunkBytes, 128);
      const uint64_t bd = ks_umma_desc(w1_addr + k * 2 * B_LBO, B_LBO, 128);
      ks_umma_bf16(d1, ad, bd, idesc, k > 0 ? 1u : 0u);
    }
    ks_umma_commit(bars + BAR_MMA1 + buf);
  };

  for (int b = 0; b < p.n_buckets; ++b) {
    const Range tr = bucket_range(tm, b, t_lo, t_hi);
    if (tr.lo >= tr.hi) continue;
    if (q > 0u) {                                   // every MMA that reads the previous family's weights is done
      ks_umma_commit(bars + BAR_DRAIN);
      ks_mbar_wait_backoff(bars + BAR_DRAIN, dphase);
      dphase ^= 1u;
    }
    ks_mbar_expect_tx(bars + BAR_W, (uint32_t)(C::W1_BYTES + C::W2_BYTES));
    ks_bulk_g2s(smem + C::OFF_W1, p.head[b].w1_img, C::W1_BYTES, bars + BAR_W);
    for (int off = 0; off < C::W2_BYTES; off += 32768) {
      const int len = C::W2_BYTES - off < 32768 ? C::W2_BYTES - off : 32768;
      ks_bulk_g2s(smem + C::OFF_W2 + off, reinterpret_cast<const char*>(p.head[b].w2_img) + off, len, bars + BAR_W);
    }
    ks_mbar_wait_backoff(bars + BAR_W, wphase);
    wphase ^= 1u;
    const uint32_t q0 = q;
    const uint32_t q1 = q0 + (uint32_t)(tr.hi - tr.lo) * (uint32_t)p.n_specs;
    // D1[0], D1[1] are free here: every a2_full of the previous family was waited for before its MMA2
    mma1(q0);
    if (q0 + 1u < q1) mma1(q0 + 1u);
    for (q = q0; q < q1; ++q) {
      if (q + 2u < q1) {                            // the short layer-1 MMA goes first: EPI1 never waits for MMA2
        ks_mbar_wait_backoff(bars + BAR_D1_FREE + (q & 1u), (q >> 1) & 1u);
        mma1(q + 2u);
      }
      mma2(q);
    }
  }
}

template <int NIN, int H>
__global__ void __launch_bounds__(kWsThreads, 1)
ks_mlp_ws_kernel(const __grid_constant__ KsMlpParams p) {
  using C = WsCfg<NIN, H>;
  extern __shared__ __align__(1024) unsigned char smem[];
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::OFF_BAR);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + BAR_COUNT);
  TileMap* tmp = reinterpret_cast<TileMap*>(smem + C::OFF_BAR + 160);
  const int tid = threadIdx.x;
  const int warp = tid >> 5;

  ks_launch_dependents();     // the step kernel's launch overlaps this kernel (it waits for our completion itself) ...
  cudaGridDependencySynchronize();   // ... as we wait for the kernel before us (ks_launch_pdl)
  if (tid == 32) tile_map_init(p, tmp);
  if (tid == 0) {
    ks_mbar_init(bars + BAR_W, 1);
    ks_mbar_init(bars + BAR_DRAIN, 1);
    for (int i = 0; i < kA2Bufs; ++i) {
      ks_mbar_init(bars + BAR_A2_FULL + i, 128);
      ks_mbar_init(bars + BAR_A2_FREE + i, 1);
    }
    for (int i = 0; i < 2; ++i) {
      ks_mbar_init(bars + BAR_A1_FULL + i, 128);
      ks_mbar_init(bars + BAR_MMA1 + i, 1);
      ks_mbar_init(bars + BAR_MMA2 + i, 1);
      ks_mbar_init(bars + BAR_D2_FREE + i, 128);
      ks_mbar_init(bars + BAR_D1_FREE + i, 128);
    }
    ks_fence_mbar_init();
  }
  if (warp == 0) { ks_tmem_alloc(tmem_slot, C::TMEM_COLS); ks_tmem_relinquish(); }
  if (tid < 128) {   // constant ones-block: K chunk 0 = {1, 1, 0, ...} per row, K chunk 1 = 0
    *reinterpret_cast<uint4*>(smem + C::OFF_ONES + tid * 16) = make_uint4(0x3F803F80u, 0u, 0u, 0u);
    *reinterpret_cast<uint4*>(smem + C::OFF_ONES + kChunkBytes + tid * 16) = make_uint4(0u, 0u, 0u, 0u);
  }
  for (int i = tid; i < p.n_buckets * H; i += kWsThreads)       // layer-3 weights of every family
    reinterpret_cast<float*>(smem + C::OFF_W3)[i] = __ldg(p.head[i / H].w3 + (i % H));
  ks_fence_proxy_async();
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
        case KS_FAM_GEMM: producer_bucket<NIN, H, KS_FAM_GEMM>(p, tm, b, tr, smem, bars, q); break;
        case KS_FAM_GROUPED_GEMM: producer_bucket<NIN, H, KS_FAM_GROUPED_GEMM>(p, tm, b, tr, smem, bars, q); break;
        case KS_FAM_ATTN: producer_bucket<NIN, H, KS_FAM_ATTN>(p, tm, b, tr, smem, bars, q); break;
        default: producer_bucket<NIN, H, KS_FAM_ELEMWISE>(p, tm, b, tr, smem, bars, q); break;
      }
    }
  } else if (warp < kProducerWarps + kEpiWarps) {
    if (p.gelu_mode == 0) epi1_items<NIN, H, 0>(p, (uint32_t)(t_hi - t_lo) * (uint32_t)p.n_specs, smem, bars, tmem_base);
    else epi1_items<NIN, H, 1>(p, (uint32_t)(t_hi - t_lo) * (uint32_t)p.n_specs, smem, bars, tmem_base);
  } else if (warp < kMmaWarp) {
    // four copies of the role, one runs: the ensemble bookkeeping stays out of the single-head loop
    if (p.any_ens) {
      if (p.gelu_mode == 0) epi2_all<NIN, H, 0, true>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
      else epi2_all<NIN, H, 1, true>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
    } else {
      if (p.gelu_mode == 0) epi2_all<NIN, H, 0, false>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
      else epi2_all<NIN, H, 1, false>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
    }
  } else if (__shfl_sync(0xffffffffu, warp, 0) == kMmaWarp) {   // warp-uniform branch, then one elected lane
    if (ks_elect_one()) mma_all<NIN, H>(p, tm, t_lo, t_hi, smem, bars, tmem_base);
  }
  ks_tc_fence_before();
  __syncthreads();
  if (warp == 0) ks_tmem_dealloc(tmem_base, C::TMEM_COLS);
}

template <int NIN, int H>
cudaError_t launch_ws(const KsMlpParams& p, int num_sms, cudaStream_t st) {
  using C = WsCfg<NIN, H>;
  const int total = p.tile_begin[p.n_buckets];
  if (total <= 0) return cudaSuccess;
  const int grid = total < num_sms ? total : num_sms;
  auto kern = ks_mlp_ws_kernel<NIN, H>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  return ks_launch_pdl(kern, grid, kWsThreads, C::SMEM_BYTES, st, p);
}

}  // namespace

cudaError_t ks_launch_mlp_ws(const KsMlpParams& p, int n_in, int h, int num_sms, cudaStream_t st) {
#define KS_CASE(NI, HH) \
  if (n_in == NI && h == HH) return launch_ws<NI, HH>(p, num_sms, st);
  KS_CASE(8, 64) KS_CASE(8, 128) KS_CASE(12, 64) KS_CASE(12, 128) KS_CASE(32, 64) KS_CASE(32, 128)
#undef KS_CASE
  return cudaErrorInvalidValue;
}
