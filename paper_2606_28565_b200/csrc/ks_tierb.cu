// ks_tierb.cu — Tier B for the GEMM and attention families (S1, S2, S4b, S5 of DESIGN.md §1): decode +
// roofline + wave quantization, trilinear interpolation of the measured-efficiency grid (Q5),
// launch floor (Eq. 2).  ONE persistent launch prices every Tier-B bucket of a call.
//
// The op moves 16 bytes per query (three int32 columns in, one fp32 latency out), so its roofline is HBM;
// what stands between the kernel and that roofline is the instruction count per query and the eight
// random shared-memory gathers.  Design:
//  * one 1024-thread CTA per SM (the grid, <= 128 KiB plus a zero tail, fills the SM's shared memory); the CTAs are
//    shared out among the buckets in proportion to their 4096-row tiles (no CTA serves two buckets), each takes a
//    contiguous tile range of its bucket and stages that bucket's grid with 1-D TMA bulk copies issued by one
//    thread, and everything that does not need the grid — column loads, decode, roofline, the interpolation
//    coordinates — runs under them;
//  * a thread owns 4 consecutive rows (16-byte column loads / latency stores, streaming cache hints) and
//    the next tile's columns are requested before the current tile is computed;
//  * floating-point work runs as packed fp32 pairs over two rows (FADD2 / FMUL2 / FFMA2: one issue slot
//    for two rows) and nothing but the int->float conversions, lg2 and rcp touches the 16-lane XU pipe:
//      - log2 v = exponent + lg2.approx(mantissa); the exponent enters as the float 2^23 + E built with one
//        LEA.HI, and (2^23 + E) - (2^23 + 127 + round(lo)) is exact, the remainder lo - round(lo) rides in the
//        coordinate's FMA: the coordinate keeps the MUFU's 2^-22 absolute error at any magnitude;
//      - the clamp to [0, dims - 1] is ONE integer instruction on the float's bits (VIMNMX.RELU);
//      - floor(c) is one FADD2.RM against 2^23 (the integer lands in the low mantissa bits), and the
//        shared-memory address is three IMADs on those bits — no F2I, no I2F;
//      - at c = dims - 1 the lower node is the last node and f = 0 exactly: the corners one node past an axis are
//        read (the next row / plane, or the zero tail behind the grid) with weight zero, no second clamp;
//  * the grid's hull test of density routing (Q16) appends out-of-hull rows with one atomic
//    per warp and tile.
// Where it stands (profiles/README.md): 0.53 of the HBM copy rate at large sizes, ~120 instructions and
// eight random 4-byte shared-memory gathers (3.8 wavefronts each) per query; a control run against conflict-free
// 2x2x2 grids gains 3 %: no single pipe bounds it, the warps' gather and arithmetic phases load the pipes in turn.
#include "ks_internal.h"
#include "ks_ptx.cuh"

namespace {

struct F2 { float x, y; };
KS_DEV F2 mk2(float a, float b) { F2 r; r.x = a; r.y = b; return r; }
KS_DEV F2 bc2(float a) { return mk2(a, a); }
KS_DEV F2 add2(F2 a, F2 b) { F2 r; ks_add2(r.x, r.y, a.x, a.y, b.x, b.y); return r; }
KS_DEV F2 mul2(F2 a, F2 b) { F2 r; ks_mul2(r.x, r.y, a.x, a.y, b.x, b.y); return r; }
KS_DEV F2 fma2(F2 a, F2 b, F2 c) { F2 r; ks_fma2(r.x, r.y, a.x, a.y, b.x, b.y, c.x, c.y); return r; }
KS_DEV F2 sub2(F2 a, F2 b) { return fma2(b, bc2(-1.0f), a); }    // a - b, exact like FADD (packed adds take no negation)
KS_DEV F2 max2(F2 a, F2 b) { return mk2(fmaxf(a.x, b.x), fmaxf(a.y, b.y)); }
// a + 2^23 rounded toward -inf: for 0 <= a < 2^22 the low mantissa bits of the result hold floor(a)
KS_DEV F2 floor_magic2(F2 a) {
  F2 r;
  asm("{\n\t.reg .b64 ra, rb, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %4};\n\t"
      "add.rm.f32x2 rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}"
      : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(8388608.0f));
  return r;
}
KS_DEV float lds_f32(uint32_t addr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
  return v;
}
KS_DEV float lds_f32_4(uint32_t addr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1+4];" : "=f"(v) : "r"(addr));
  return v;
}

template <bool F32>
KS_DEV void load_rows4(const KsBucketDev& bk, int row0, int n, int (&v)[4][3]) {
  if (row0 + 4 <= n) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
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
      for (int c = 0; c < 3; ++c) v[j][c] = (row0 + j < n) ? ks_load_col(bk.cols[c], row0 + j, F32) : 0;
  }
}

template <typename T>
KS_DEV void store4(T* base, long long off, int row0, int n, T a, T b, T c, T d) {
  T* ptr = base + off + row0;
  if (((off & 3ll) == 0) && row0 + 4 <= n) {
    float4 q;
    q.x = *reinterpret_cast<float*>(&a); q.y = *reinterpret_cast<float*>(&b);
    q.z = *reinterpret_cast<float*>(&c); q.w = *reinterpret_cast<float*>(&d);
    __stcs(reinterpret_cast<float4*>(ptr), q);
  } else {
    if (row0 + 0 < n) ptr[0] = a;
    if (row0 + 1 < n) ptr[1] = b;
    if (row0 + 2 < n) ptr[2] = c;
    if (row0 + 3 < n) ptr[3] = d;
  }
}

// The three axis values of a row as non-negative ints and as floats (Q5: GEMM (M, N, K);
// attention (batch, q_len, max(kv_len, q_len))).  Both families decode from exactly these.
struct Axes2 {
  int i[3][2];
  F2 f[3];
};
template <int FAM>
KS_DEV Axes2 axes_of(const int* va, const int* vb) {
  Axes2 a;
#pragma unroll
  for (int k = 0; k < 3; ++k) { a.i[k][0] = ks_nonneg(va[k]); a.i[k][1] = ks_nonneg(vb[k]); }
  if (FAM == KS_FAM_ATTN) {
    a.i[2][0] = max(a.i[2][0], a.i[1][0]);
    a.i[2][1] = max(a.i[2][1], a.i[1][1]);
  }
#pragma unroll
  for (int k = 0; k < 3; ++k) a.f[k] = mk2((float)a.i[k][0], (float)a.i[k][1]);
  return a;
}

// spec-independent work terms of a row pair: F_comp, F_mem / s
template <int FAM>
KS_DEV void work_of(const Axes2& a, const KsBucketDev& bk, F2& F, F2& Ys) {
  if (FAM == KS_FAM_GEMM) {
    const F2 mn = mul2(a.f[0], a.f[1]);
    F = mul2(mn, add2(a.f[2], a.f[2]));                         // 2 M N K
    Ys = fma2(a.f[0], a.f[2], fma2(a.f[2], a.f[1], mn));        // M K + K N + M N
  } else {
    // causal pairs: cached history + own triangle: q (kv - q) + q (q + 1) / 2
    const F2 q = a.f[1], kv = a.f[2];
    const F2 pairs = fma2(q, sub2(kv, q), mul2(mul2(q, bc2(0.5f)), add2(q, bc2(1.0f))));
    const float c1 = 4.0f * (float)bk.hq * (float)bk.hd;
    F = mul2(mul2(a.f[0], bc2(c1)), pairs);                     // 4 B Hq d pairs
    const F2 g = fma2(q, bc2((float)bk.hq), mul2(kv, bc2((float)bk.hkv)));
    Ys = mul2(mul2(a.f[0], bc2(2.0f * (float)bk.hd)), g);       // 2 B d (q Hq + kv Hkv)
  }
}

// ceil(a / d) for 1 <= a < 2^31 as floor((a - 1) / d) + 1: four instructions (a = 0 gives garbage: callers zero it)
KS_DEV uint32_t cdiv_pos(uint32_t a, const KsFastDiv& f) { return (__umulhi(2u * a - 2u, f.mul) >> f.shr) + 1u; }

template <int FAM>
KS_DEV uint32_t tiles_of(const Axes2& a, int j, const KsBucketDev& bk, const KsSpecDev& sp) {
  if (FAM == KS_FAM_GEMM) {
    const uint32_t B = ks_sat31((unsigned long long)cdiv_pos(a.i[0][j], sp.tile_m) * cdiv_pos(a.i[1][j], sp.tile_n));
    return (a.i[0][j] == 0 || a.i[1][j] == 0) ? 0u : B;
  }
  const uint32_t B = ks_sat31((unsigned long long)a.i[0][j] * (unsigned long long)bk.hq * cdiv_pos(a.i[1][j], sp.tile_m));
  return a.i[1][j] == 0 ? 0u : B;
}

// Eq. 2's roofline with wave quantization for a row pair: t_roof = max(F/P u, Y/BW)
KS_DEV F2 roof2(F2 F, F2 Ys, const uint32_t (&B)[2], uint32_t (&W)[2], float s, const KsSpecDev& sp) {
  W[0] = cdiv_pos(B[0], sp.slots);                                // (B = 0 is overridden below)
  W[1] = cdiv_pos(B[1], sp.slots);
  const F2 rB = mk2(__fdividef(1.0f, (float)B[0]), __fdividef(1.0f, (float)B[1]));
  const F2 u = mul2(mul2(mk2((float)W[0], (float)W[1]), bc2(sp.slots_f)), rB);
  const F2 tcu = mul2(mul2(F, bc2(sp.inv_peak_flops)), u);
  const F2 tm = mul2(Ys, bc2(s * sp.inv_peak_bw));
  F2 t = max2(tcu, tm);
  if (B[0] == 0u) { t.x = 0.0f; W[0] = 0u; }
  if (B[1] == 0u) { t.y = 0.0f; W[1] = 0u; }
  return t;
}

// (a & b) | c in one LOP3 (the constants stay in registers: with immediates it takes two)
KS_DEV uint32_t and_or(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t d;
  asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}
// clamp a float to [0, hi] (hi >= 0) with ONE integer instruction: non-negative floats order like their bit
// patterns and every negative float is a negative int, so max(min(bits, bits(hi)), 0) is the clamp (VIMNMX.RELU)
KS_DEV float clamp0(float c, float hi) { return __int_as_float(__vimin_s32_relu(__float_as_int(c), __float_as_int(hi))); }

// interpolation coordinates of a row pair along one axis: fractional part f and the magic float whose
// low mantissa bits hold the lower node index.  c = clamp((log2 v - lo) * scale, 0, top) (Q5).  At
// c = top the lower node IS the last node and f = 0 exactly, so the "upper" corners (one node past the axis:
// the next row / plane, or the zero padding behind the grid) enter with weight zero — no min() against
// dims - 2 is needed.
KS_DEV void coord2(F2 vf, const KsTierBGrid& g, int a, uint32_t mant_mask, uint32_t one_bits, F2& frac, F2& tmag) {
  const uint32_t b0 = __float_as_uint(vf.x), b1 = __float_as_uint(vf.y);
  // 2^23 + E (E = biased exponent; v = 0 gives E = 0, far below any span: clamps to the first node)
  const F2 ex = mk2(__uint_as_float((b0 >> 23) | 0x4B000000u), __uint_as_float((b1 >> 23) | 0x4B000000u));
  const F2 lm = mk2(__log2f(__uint_as_float(and_or(b0, mant_mask, one_bits))),
                    __log2f(__uint_as_float(and_or(b1, mant_mask, one_bits))));
  const F2 x = add2(add2(ex, bc2(g.nkc[a])), lm);                 // log2 v - round(lo) (first add exact)
  const F2 cu = fma2(x, bc2(g.scale[a]), bc2(g.nrs[a]));
  const F2 c = mk2(clamp0(cu.x, g.top[a]), clamp0(cu.y, g.top[a]));
  tmag = floor_magic2(c);
  frac = sub2(c, add2(tmag, bc2(-8388608.0f)));
}

template <int FAM, bool F32, bool ONE, int NT>
KS_DEV void run_bucket(const KsTierBParams& p, const int b, const int tile0, const int tile1, const uint32_t sgrid,
                       uint64_t* bar, const uint32_t parity) {
  const KsBucketDev& bk = p.bk[b];
  const KsTierBGrid& g = p.grid[b];
  const int n = bk.n;
  const float s = (float)bk.s;
  // shared-memory byte address of node (i0, i1, i2) = kbase + sum_a bits(2^23 + i_a) * 4 stride_a
  const uint32_t kbase = sgrid - 0x4B000000u * (uint32_t)(g.stride4[0] + g.stride4[1] + g.stride4[2]);
  uint32_t mant_mask = 0x007fffffu, one_bits = 0x3f800000u;
  asm volatile("" : "+r"(mant_mask), "+r"(one_bits));            // keep them in registers (see and_or)
  bool grid_ready = false;
  int row0 = (tile0 - p.tile_begin[b]) * (NT * 4) + (int)threadIdx.x * 4;
  int nxt[4][3];
  load_rows4<F32>(bk, row0, n, nxt);
#pragma unroll 1
  for (int tile = tile0; tile < tile1; ++tile) {
    int v[4][3];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int c = 0; c < 3; ++c) v[j][c] = nxt[j][c];
    const int cur0 = row0;
    row0 += NT * 4;
    if (tile + 1 < tile1) load_rows4<F32>(bk, row0, n, nxt);      // next tile's columns fly under this tile's math
    if (g.route_idx != nullptr) {                                 // (all 32 lanes vote: rows past the end count as inside)
      // density routing, pass 1 (Q16): rows outside the measured hull are listed for the learned
      // head, which overwrites their clamped Tier-B value afterwards.  One atomic per warp.
      unsigned out[4];
      int cnt = 0;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const long long a0 = v[j][0], a1 = v[j][1], a2 = (FAM == KS_FAM_ATTN && v[j][2] < v[j][1]) ? v[j][1] : v[j][2];
        const bool in = a0 >= g.vmin[0] && a0 <= g.vmax[0] && a1 >= g.vmin[1] && a1 <= g.vmax[1] && a2 >= g.vmin[2] && a2 <= g.vmax[2];
        out[j] = __ballot_sync(0xffffffffu, cur0 + j < n && !in);
        cnt += __popc(out[j]);
      }
      if (cnt) {                                                  // warp-uniform
        const unsigned lane = threadIdx.x & 31u, below = (1u << lane) - 1u;
        int base = 0;
        if (lane == 0) base = atomicAdd(g.route_count, cnt);
        base = __shfl_sync(0xffffffffu, base, 0);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if ((out[j] >> lane) & 1u) g.route_idx[base + __popc(out[j] & below)] = cur0 + j;
          base += __popc(out[j]);
        }
      }
    }

    if (cur0 >= n) continue;

    // ---- everything that does not need the grid
    F2 fr[2][3];
    uint32_t addr[4];
    F2 Fw[2], Yw[2];
    Axes2 ax[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      ax[h] = axes_of<FAM>(v[2 * h], v[2 * h + 1]);
      work_of<FAM>(ax[h], bk, Fw[h], Yw[h]);
      uint32_t a0 = kbase, a1 = kbase;
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        F2 tmag;
        coord2(ax[h].f[a], g, a, mant_mask, one_bits, fr[h][a], tmag);
        a0 += __float_as_uint(tmag.x) * (uint32_t)g.stride4[a];
        a1 += __float_as_uint(tmag.y) * (uint32_t)g.stride4[a];
      }
      addr[2 * h] = a0;
      addr[2 * h + 1] = a1;
    }
    if (!grid_ready) { ks_mbar_wait(bar, parity); grid_ready = true; }

    // ---- eight gathers and seven lerps per row (blend along axis 2, then 1, then 0, of the stored e)
    float e[4];
    const uint32_t s0 = (uint32_t)g.stride4[0], s1 = (uint32_t)g.stride4[1];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      F2 c[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t o = (k & 2 ? s0 : 0u) + (k & 1 ? s1 : 0u);
        const uint32_t pa = addr[2 * h] + o, pb = addr[2 * h + 1] + o;
        const F2 lo = mk2(lds_f32(pa), lds_f32(pb)), hi = mk2(lds_f32_4(pa), lds_f32_4(pb));
        c[k] = fma2(fr[h][2], sub2(hi, lo), lo);
      }
      const F2 c0 = fma2(fr[h][1], sub2(c[1], c[0]), c[0]);
      const F2 c1 = fma2(fr[h][1], sub2(c[3], c[2]), c[2]);
      const F2 r = fma2(fr[h][0], sub2(c1, c0), c0);
      e[2 * h] = fmaxf(r.x, 0.0009765625f);                      // guard e >= 2^-10 (Q3)
      e[2 * h + 1] = fmaxf(r.y, 0.0009765625f);
    }

    // ---- Eq. 2 per spec: t = max(t_roof / e, t0)
    const int n_specs = ONE ? 1 : p.n_specs;
#pragma unroll 1
    for (int sidx = 0; sidx < n_specs; ++sidx) {
      const KsSpecDev& sp = p.specs.s[ONE ? 0 : sidx];
      const long long off = (long long)sidx * n;
      float t[4], tr[4];
      uint32_t B[4], W[4];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        uint32_t Bp[2] = {tiles_of<FAM>(ax[h], 0, bk, sp), tiles_of<FAM>(ax[h], 1, bk, sp)}, Wp[2];
        const F2 troof = roof2(Fw[h], Yw[h], Bp, Wp, s, sp);
        B[2 * h] = Bp[0]; B[2 * h + 1] = Bp[1];
        W[2 * h] = Wp[0]; W[2 * h + 1] = Wp[1];
        tr[2 * h] = troof.x; tr[2 * h + 1] = troof.y;
        t[2 * h] = fmaxf(__fdividef(troof.x, e[2 * h]), sp.t0);
        t[2 * h + 1] = fmaxf(__fdividef(troof.y, e[2 * h + 1]), sp.t0);
      }
      store4<float>(bk.lat, off, cur0, n, t[0], t[1], t[2], t[3]);
      if (bk.tiles) store4<int>(bk.tiles, off, cur0, n, (int)B[0], (int)B[1], (int)B[2], (int)B[3]);
      if (bk.waves) store4<int>(bk.waves, off, cur0, n, (int)W[0], (int)W[1], (int)W[2], (int)W[3]);
      if (bk.troof) store4<float>(bk.troof, off, cur0, n, tr[0], tr[1], tr[2], tr[3]);
    }
  }
  if (!grid_ready) ks_mbar_wait(bar, parity);                     // never leave a bulk copy in flight behind us
}

template <bool F32, bool ONE, int NT>
__global__ void __launch_bounds__(NT, 1) ks_tierb_kernel(const __grid_constant__ KsTierBParams p) {
  ks_launch_dependents();     // the next kernel of the stream may be scheduled now (it waits for us itself) ...
  extern __shared__ __align__(128) float sgrid_f[];
  __shared__ __align__(8) uint64_t bar;
  const uint32_t sgrid = ks_smem_u32(sgrid_f);
  if (threadIdx.x == 0) { ks_mbar_init(&bar, 1); ks_fence_mbar_init(); }
  __syncthreads();

  // The launcher gave every bucket a share of the CTAs in proportion to its tiles (no CTA serves two
  // buckets: it would stage a second grid in the middle of its range); inside a bucket, contiguous tile ranges.
  int b = 0;
  while (b + 1 < p.n_buckets && (int)blockIdx.x >= p.cta_begin[b + 1]) ++b;
  const long long lc = (int)blockIdx.x - p.cta_begin[b], nc = p.cta_begin[b + 1] - p.cta_begin[b];
  const long long tiles = p.tile_begin[b + 1] - p.tile_begin[b];
  const int t0 = p.tile_begin[b] + (int)(tiles * lc / nc), t1 = p.tile_begin[b] + (int)(tiles * (lc + 1) / nc);
  if (threadIdx.x == 0) {
    const uint32_t bytes = (uint32_t)p.grid[b].bytes;
    ks_mbar_expect_tx(&bar, bytes);
    for (uint32_t o = 0; o < bytes; o += 32768u)
      ks_bulk_g2s(reinterpret_cast<char*>(sgrid_f) + o, reinterpret_cast<const char*>(p.grid[b].values) + o,
                  min(32768u, bytes - o), &bar);
  }
  // ... as we wait for the one before us (ks_launch_pdl) -- AFTER the grid's bulk copies have been issued: the grid is
  // model data that ks_load_grid copied in synchronously, nothing on the stream writes it, so its staging (128 KiB per
  // CTA) may overlap the tail of the preceding kernel; descriptor columns and outputs are touched only below
  cudaGridDependencySynchronize();
  if (p.bk[b].family == KS_FAM_GEMM) run_bucket<KS_FAM_GEMM, F32, ONE, NT>(p, b, t0, t1, sgrid, &bar, 0u);
  else run_bucket<KS_FAM_ATTN, F32, ONE, NT>(p, b, t0, t1, sgrid, &bar, 0u);
}

}  // namespace

cudaError_t ks_launch_tierb(const KsTierBParams& p, int num_sms, cudaStream_t st) {
  const bool one = p.n_specs == 1;
  const int nt = one ? 1024 : 512;                                // the spec loop keeps more state per row: 128 registers
  KsTierBParams q = p;
  bool f32 = false;
  int max_bytes = 0;
  q.tile_begin[0] = 0;
  for (int b = 0; b < q.n_buckets; ++b) {
    q.tile_begin[b + 1] = q.tile_begin[b] + (q.bk[b].n + nt * 4 - 1) / (nt * 4);
    f32 = q.bk[b].col_f32 != 0;                                   // (the caller groups buckets of one column type)
    max_bytes = q.grid[b].bytes > max_bytes ? q.grid[b].bytes : max_bytes;
  }
  const int total = q.tile_begin[q.n_buckets];
  if (total == 0) return cudaSuccess;
  // persistent: one CTA per SM, shared out among the buckets in proportion to their tiles (at least one each,
  // never more than a bucket has tiles)
  int share[KS_TIERB_MAX_BUCKETS], tb[KS_TIERB_MAX_BUCKETS], blocks = 0;
  for (int b = 0; b < q.n_buckets; ++b) {
    tb[b] = q.tile_begin[b + 1] - q.tile_begin[b];
    share[b] = (int)((long long)num_sms * tb[b] / total);
    share[b] = share[b] < 1 ? 1 : share[b];
    share[b] = share[b] > tb[b] ? tb[b] : share[b];
    blocks += share[b];
  }
  for (;;) {                                                      // hand out what the rounding left (or took too much)
    int hi = -1, lo = -1;
    for (int b = 0; b < q.n_buckets; ++b) {
      if (share[b] < tb[b] && (hi < 0 || (long long)tb[b] * share[hi] > (long long)tb[hi] * share[b])) hi = b;
      if (share[b] > 1 && (lo < 0 || (long long)tb[b] * share[lo] < (long long)tb[lo] * share[b])) lo = b;
    }
    if (blocks < num_sms && hi >= 0) { ++share[hi]; ++blocks; }
    else if (blocks > num_sms && lo >= 0) { --share[lo]; --blocks; }
    else break;
  }
  q.cta_begin[0] = 0;
  for (int b = 0; b < q.n_buckets; ++b) q.cta_begin[b + 1] = q.cta_begin[b] + share[b];
  const size_t smem = (size_t)max_bytes;
  void (*kern)(const KsTierBParams) =
      one ? (f32 ? ks_tierb_kernel<true, true, 1024> : ks_tierb_kernel<false, true, 1024>)
          : (f32 ? ks_tierb_kernel<true, false, 512> : ks_tierb_kernel<false, false, 512>);
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  return ks_launch_pdl(kern, blocks, nt, smem, st, q);
}
