/* ks_oracle.c — CPU ORACLE (test infrastructure only; see ks_oracle.h).
 * Plain C99, double precision, one descriptor at a time, no blocking/fusion/SIMD.
 * Every function cites the PAPER.md passage or the DESIGN.md reading it follows.
 */
#include "ks_oracle.h"
#include <math.h>
#include <stddef.h>

/* ---------------------------------------------------------------- small helpers */
static int64_t nonneg(int64_t v) { return v > 0 ? v : 0; }
static int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }
static double clip1(double x) { return x < -1.0 ? -1.0 : (x > 1.0 ? 1.0 : x); }
static double dmax(double a, double b) { return a > b ? a : b; }
static double dmin(double a, double b) { return a < b ? a : b; }

/* bfloat16 = 1 sign, 8 exponent, 7 stored mantissa bits -> 8 significant bits.
 * Round to nearest, ties to even (rint under the default rounding mode). DESIGN.md Q11. */
double kso_bf16(double x) {
  if (x == 0.0 || isnan(x) || isinf(x)) return x;
  int e;
  double m = frexp(x, &e);          /* x = m 2^e, 0.5 <= |m| < 1 */
  int keep = 8;
  if (e < -125) keep = 8 - (-125 - e); /* bf16 subnormals (min normal 2^-126) */
  if (keep <= 0) {
    /* below half the smallest subnormal rounds to 0; exactly representable cases handled by rint */
    double q = ldexp(x, 133);       /* smallest subnormal is 2^-133 */
    return ldexp(rint(q), -133);
  }
  return ldexp(rint(ldexp(m, keep)), e - keep);
}

/* GELU, exact erf form (Q6; layer sizes/activations come from BASELINE.json) */
double kso_gelu(double x) { return 0.5 * x * (1.0 + erf(x / sqrt(2.0))); }
double kso_sigmoid(double z) { return 1.0 / (1.0 + exp(-z)); }

/* heads are trained against log eta = log(t_meas / t_roof); eta >= 1 (the roofline is a
 * lower bound), so a negative output is floored at log eta = 0 (Q21). */
double kso_eta_from_log(double z) { return exp(z > 0.0 ? z : 0.0); }

/* ---------------------------------------------------------------- S1: F_comp, F_mem, B
 * PAPER.md:193 names "the kernel's FLOPs and bytes" without printing formulas; Q1. */

/* a prefill chunk attends "its cached history plus its own causal triangle":
 * query i (1-based within the chunk) sees hist + i keys  ->  q*hist + q(q+1)/2 pairs. */
int64_t kso_attn_pairs(int64_t q, int64_t kv) {
  q = nonneg(q);
  if (kv < q) kv = q;
  int64_t hist = kv - q;
  return q * hist + q * (q + 1) / 2;
}

/* elementwise sub-ops: RMSNorm, SiLU*Mul, RoPE, KV-write, Embedding, residual-add (Tables 2/4,
 * PAPER.md:271-283, :323-336): words read+written per element, and FLOPs per element. */
static const double EW_RW[6] = {2, 3, 2, 2, 2, 3};
static const double EW_FL[6] = {4, 4, 6, 0, 0, 1};

void kso_work(const kso_desc *d, const kso_spec *hw, double *F, double *Y, int64_t *B) {
  double s = (double)d->s;
  double f = 0, y = 0;
  int64_t b = 0;
  switch (d->family) {
  case KSO_GEMM: {
    int64_t M = nonneg(d->v[0]), N = nonneg(d->v[1]), K = nonneg(d->v[2]);
    f = 2.0 * (double)M * (double)N * (double)K;
    y = s * ((double)M * K + (double)K * N + (double)M * N);
    b = ceil_div(M, hw->tile_m) * ceil_div(N, hw->tile_n);
    break;
  }
  case KSO_GROUPED: {
    int64_t N = nonneg(d->v[0]), K = nonneg(d->v[1]);
    int64_t sum = 0, act = 0;
    for (int e = 0; e < KSO_EXPERTS; ++e) {
      int64_t m = nonneg(d->v[2 + e]);
      sum += m;
      if (m > 0) act += 1;
      b += ceil_div(m, hw->tile_m) * ceil_div(N, hw->tile_n);
    }
    f = 2.0 * (double)N * (double)K * (double)sum;
    y = s * ((double)K * sum + (double)act * K * N + (double)N * sum);
    break;
  }
  case KSO_ATTN: {
    int64_t Bq = nonneg(d->v[0]), q = nonneg(d->v[1]), kv = nonneg(d->v[2]);
    if (kv < q) kv = q;
    double pairs = (double)kso_attn_pairs(q, kv);
    f = 4.0 * (double)Bq * (double)d->hq * (double)d->d * pairs;       /* QK^T and PV: 2 x 2 FLOP/pair/dim */
    y = s * (2.0 * (double)Bq * q * d->hq * d->d                      /* Q read, O written */
             + 2.0 * (double)Bq * kv * d->hkv * d->d);                /* K, V read */
    b = Bq * d->hq * ceil_div(q, hw->tile_m);
    break;
  }
  case KSO_ELEMWISE: {
    int64_t n = nonneg(d->v[0]);
    int64_t op = d->v[1];
    if (op < 0) op = 0;
    if (op > 5) op = 5;
    y = s * (double)n * EW_RW[op];
    f = (double)n * EW_FL[op];
    b = ceil_div(n, hw->ew_elems_per_cta);
    break;
  }
  default: break;
  }
  if (b == 0) { f = 0; y = 0; }   /* nothing is launched */
  *F = f; *Y = y; *B = b;
}

/* ---------------------------------------------------------------- S2: wave quantization
 * PAPER.md:88 (Fig. 2): u = ceil(B/N_SM) N_SM / B >= 1. DESIGN.md Q4: slots S = N_SM x CTAs/SM. */
void kso_wave(int64_t B, int64_t S, int64_t *W, double *u) {
  if (B <= 0) { *W = 0; *u = 1.0; return; }
  *W = ceil_div(B, S);
  *u = (double)(*W) * (double)S / (double)B;
}

/* PAPER.md:191 Eq. 2: t_roof = max(F_comp/P_peak * u, F_mem/BW_peak) */
void kso_roofline(const kso_desc *d, const kso_spec *hw, kso_roof *r) {
  kso_work(d, hw, &r->F, &r->Y, &r->B);
  kso_wave(r->B, hw->n_sm * hw->ctas_per_sm, &r->W, &r->u);
  r->t_comp = r->F / hw->peak_flops;
  r->t_mem = r->Y / hw->peak_bw;
  r->t_roof = dmax(r->t_comp * r->u, r->t_mem);
}

/* ---------------------------------------------------------------- S3: features
 * "arithmetic intensity and its position relative to the roofline ridge, per-SM
 * work and occupancy, wave count, and L2 cache residency".  Exact list: DESIGN.md Q2. */
void kso_features(const kso_desc *d, const kso_spec *hw, const kso_roof *r, int n_in, double *x) {
  for (int i = 0; i < n_in; ++i) x[i] = 0.0;
  if (r->B <= 0) return;
  double S = (double)(hw->n_sm * hw->ctas_per_sm);
  double AI = dmax(r->F / r->Y, ldexp(1.0, -10));
  double ridge = hw->peak_flops / hw->peak_bw;
  x[0] = clip1(log2(AI) / 16.0);                                       /* AI */
  x[1] = clip1(log2(AI / ridge) / 16.0);                               /* AI relative to the ridge */
  x[2] = clip1(log2((double)r->W) / 16.0);                             /* wave count */
  x[3] = (double)r->B / ((double)r->W * S);                            /* occupancy incl. last wave = 1/u */
  x[4] = clip1(log2(dmax(r->t_roof / hw->t0, ldexp(1.0, -10))) / 16.0);/* body vs launch floor */
  x[5] = dmin(1.0, hw->l2_bytes / r->Y);                               /* L2 residency */
  x[6] = clip1(log2(dmax(r->t_comp * r->u / r->t_mem, ldexp(1.0, -20))) / 20.0); /* signed ridge distance */
  x[7] = clip1(log2(dmax((double)r->B / S, ldexp(1.0, -10))) / 16.0);  /* per-slot work */
  if (n_in <= 8) return;
  double lg1 = 1.0;                                                    /* log2 of max(.,1) */
  switch (d->family) {
  case KSO_GEMM:
    x[8] = clip1(log2(dmax((double)d->v[0], lg1)) / 16.0);
    x[9] = clip1(log2(dmax((double)d->v[1], lg1)) / 16.0);
    x[10] = clip1(log2(dmax((double)d->v[2], lg1)) / 16.0);
    break;
  case KSO_GROUPED: {
    double sum = 0;
    for (int e = 0; e < KSO_EXPERTS; ++e) sum += (double)nonneg(d->v[2 + e]);
    x[8] = clip1(log2(dmax(sum, lg1)) / 16.0);
    x[9] = clip1(log2(dmax((double)d->v[0], lg1)) / 16.0);
    x[10] = clip1(log2(dmax((double)d->v[1], lg1)) / 16.0);
    break;
  }
  case KSO_ATTN: {
    int64_t kv = d->v[2] < d->v[1] ? d->v[1] : d->v[2];
    x[8] = clip1(log2(dmax((double)d->v[0], lg1)) / 16.0);
    x[9] = clip1(log2(dmax((double)d->v[1], lg1)) / 16.0);
    x[10] = clip1(log2(dmax((double)kv, lg1)) / 16.0);
    break;
  }
  case KSO_ELEMWISE: {
    int64_t op = d->v[1] < 0 ? 0 : (d->v[1] > 5 ? 5 : d->v[1]);
    x[8] = clip1(log2(dmax((double)d->v[0], lg1)) / 32.0);
    x[9] = EW_RW[op] / 4.0;
    x[10] = EW_FL[op] / 8.0;
    break;
  }
  default: break;
  }
  x[11] = (double)d->s / 4.0;
  if (n_in <= 12) return;
  if (d->family == KSO_GROUPED) {                                      /* expert-load shape */
    double sum = 0, mx = 0, act = 0;
    for (int e = 0; e < KSO_EXPERTS; ++e) {
      double m = (double)nonneg(d->v[2 + e]);
      sum += m; if (m > mx) mx = m; if (m > 0) act += 1;
    }
    for (int e = 0; e < KSO_EXPERTS; ++e) x[12 + e] = (double)nonneg(d->v[2 + e]) / sum;
    x[20] = (mx / (sum / KSO_EXPERTS)) / 8.0;                          /* max over mean load, /8 */
    x[21] = act / KSO_EXPERTS;
  }
  /* x[22..31] = 0 */
}

/* ---------------------------------------------------------------- S4a: Tier-A head
 * PAPER.md:199-201 (per-family head; the small MLP is one pool member). Scalar triple loop. */
double kso_mlp_z(const kso_head *h, const double *x) {
  double a1[1024], a2[1024];
  for (int j = 0; j < h->h1; ++j) {
    double acc = h->b1[j];
    for (int i = 0; i < h->n_in; ++i) acc += x[i] * h->W1[(size_t)i * h->h1 + j];
    a1[j] = kso_gelu(acc);
  }
  for (int j = 0; j < h->h2; ++j) {
    double acc = h->b2[j];
    for (int i = 0; i < h->h1; ++i) acc += a1[i] * h->W2[(size_t)i * h->h2 + j];
    a2[j] = kso_gelu(acc);
  }
  double z = h->b3;
  for (int j = 0; j < h->h2; ++j) z += a2[j] * h->w3[j];
  return z;
}

/* The head's output convention: utilisation e = sigmoid(z) (Q3), or z = log eta, e = 1 / eta (Q21). */
double kso_head_e(const kso_head *h, const double *x) {
  const double z = kso_mlp_z(h, x);
  return h->log_eta ? 1.0 / kso_eta_from_log(z) : kso_sigmoid(z);
}

/* ---------------------------------------------------------------- S4b: Tier-B grid
 * "eta is obtained by interpolating this grid"; scheme/clamp: DESIGN.md Q5. */
void kso_grid_axes(const kso_desc *d, double v[3]) {
  switch (d->family) {
  case KSO_GEMM: v[0] = (double)d->v[0]; v[1] = (double)d->v[1]; v[2] = (double)d->v[2]; break;
  case KSO_GROUPED: {
    double sum = 0;
    for (int e = 0; e < KSO_EXPERTS; ++e) sum += (double)nonneg(d->v[2 + e]);
    v[0] = sum; v[1] = (double)d->v[0]; v[2] = (double)d->v[1];
    break;
  }
  case KSO_ATTN:
    v[0] = (double)d->v[0]; v[1] = (double)d->v[1];
    v[2] = (double)(d->v[2] < d->v[1] ? d->v[1] : d->v[2]);
    break;
  default: {
    int64_t op = d->v[1] < 0 ? 0 : (d->v[1] > 5 ? 5 : d->v[1]);
    v[0] = (double)d->v[0]; v[1] = ldexp(1.0, (int)op); v[2] = 1.0;
    break;
  }
  }
}

double kso_trilinear(const kso_grid *g, const double v[3]) {
  int64_t i0[3], i1[3];
  double f[3];
  for (int a = 0; a < 3; ++a) {
    int64_t dm = g->dims[a];
    if (dm <= 1) { i0[a] = 0; i1[a] = 0; f[a] = 0.0; continue; }
    double c = (v[a] > 0.0) ? (log2(v[a]) - g->lo[a]) / (g->hi[a] - g->lo[a]) * (double)(dm - 1) : 0.0;
    if (!(c > 0.0)) c = 0.0;                         /* clamp (also catches NaN) */
    if (c > (double)(dm - 1)) c = (double)(dm - 1);
    int64_t i = (int64_t)floor(c);
    if (i > dm - 2) i = dm - 2;
    i0[a] = i; i1[a] = i + 1; f[a] = c - (double)i;
  }
  const double *val = g->values;
  int64_t d1 = g->dims[1], d2 = g->dims[2];
#define AT(i, j, k) val[((i) * d1 + (j)) * d2 + (k)]
  double c00 = AT(i0[0], i0[1], i0[2]) * (1 - f[2]) + AT(i0[0], i0[1], i1[2]) * f[2];
  double c01 = AT(i0[0], i1[1], i0[2]) * (1 - f[2]) + AT(i0[0], i1[1], i1[2]) * f[2];
  double c10 = AT(i1[0], i0[1], i0[2]) * (1 - f[2]) + AT(i1[0], i0[1], i1[2]) * f[2];
  double c11 = AT(i1[0], i1[1], i0[2]) * (1 - f[2]) + AT(i1[0], i1[1], i1[2]) * f[2];
#undef AT
  double c0 = c00 * (1 - f[1]) + c01 * f[1];
  double c1 = c10 * (1 - f[1]) + c11 * f[1];
  return c0 * (1 - f[0]) + c1 * f[0];
}

/* ---------------------------------------------------------------- S5: one prediction
 * PAPER.md:191 Eq. 2: t = max(t_roof * eta, t0); eta = 1/e (Q3). */
/* PAPER.md:219 Eq. 3 */
double kso_allreduce(int64_t S, int64_t P, const kso_spec *hw) {
  if (S < 0) S = 0;
  if (P <= 1) return hw->ar_alpha0;
  return hw->ar_alpha0 + 2.0 * (double)(P - 1) / (double)P * ((double)S / hw->ar_beta_eff);
}

double kso_predict_one(const kso_desc *d, const kso_spec *hw, int tier, const kso_head *h,
                       const kso_grid *g, kso_roof *rout, double *e_out) {
  kso_roof r;
  if (d->family == KSO_ALLREDUCE) {   /* a communication row: Eq. 3 as it stands, for every tier */
    const double t = kso_allreduce(d->v[0], d->v[1], hw);
    r.F = 0.0; r.Y = 0.0; r.B = 0; r.W = 0; r.u = 1.0; r.t_comp = 0.0; r.t_mem = 0.0; r.t_roof = t;
    if (rout) *rout = r;
    if (e_out) *e_out = 1.0;
    return t;
  }
  kso_roofline(d, hw, &r);
  double e = 1.0;
  if (tier == KSO_TIER_A) {
    double x[32];
    kso_features(d, hw, &r, h->n_in, x);
    for (int i = 0; i < h->n_in; ++i) x[i] = kso_bf16(x[i]);   /* bf16 inputs, Q11 */
    e = kso_head_e(h, x);
  } else if (tier == KSO_TIER_B) {
    double v[3];
    kso_grid_axes(d, v);
    e = kso_trilinear(g, v);
  }
  if (tier != KSO_TIER_NONE) e = dmax(e, ldexp(1.0, -10));      /* guard, Q3 */
  if (rout) *rout = r;
  if (e_out) *e_out = e;
  return dmax(r.t_roof / e, hw->t0);                            /* floor applied after eta */
}

/* PAPER.md:197 Fig. 6, :201; Q15 */
double kso_bounded_e(const kso_bounded *bh, const double *x, int64_t W) {
  double zg = bh->b_gamma, za = bh->b_alpha;
  for (int i = 0; i < bh->n_in; ++i) { zg += bh->w_gamma[i] * x[i]; za += bh->w_alpha[i] * x[i]; }
  const double gamma = kso_sigmoid(zg);
  const double alpha = dmax(za, 0.0);
  double e = gamma;
  if (W > 0) e = gamma - alpha / (double)W;
  if (e > 1.0) e = 1.0;
  return dmax(e, ldexp(1.0, -10));
}

double kso_predict_one_bounded(const kso_desc *d, const kso_spec *hw, const kso_bounded *bh, kso_roof *rout,
                               double *e_out) {
  if (d->family == KSO_ALLREDUCE) return kso_predict_one(d, hw, KSO_TIER_NONE, NULL, NULL, rout, e_out);
  kso_roof r;
  kso_roofline(d, hw, &r);
  double x[32];
  kso_features(d, hw, &r, bh->n_in, x);
  const double e = kso_bounded_e(bh, x, r.W);
  if (rout) *rout = r;
  if (e_out) *e_out = e;
  return dmax(r.t_roof / e, hw->t0);
}

int kso_predict_batch_bounded(int family, int64_t n, const double *const *cols, int n_cols, int64_t s,
                              int64_t hq, int64_t hkv, int64_t dh, const kso_spec *specs, int n_specs,
                              const kso_bounded *bh, double *lat, int64_t *tiles, int64_t *waves, double *troof) {
  if (n < 0 || n_cols < 0 || n_cols > KSO_MAX_COLS || !bh) return -1;
  for (int sp = 0; sp < n_specs; ++sp) {
    for (int64_t i = 0; i < n; ++i) {
      kso_desc d;
      d.family = family; d.s = s; d.hq = hq; d.hkv = hkv; d.d = dh;
      for (int c = 0; c < KSO_MAX_COLS; ++c) d.v[c] = (c < n_cols) ? (int64_t)llround(cols[c][i]) : 0;
      kso_roof r;
      const double t = kso_predict_one_bounded(&d, &specs[sp], bh, &r, NULL);
      const size_t o = (size_t)sp * (size_t)n + (size_t)i;
      lat[o] = t;
      if (tiles) tiles[o] = r.B;
      if (waves) waves[o] = r.W;
      if (troof) troof[o] = r.t_roof;
    }
  }
  return 0;
}

/* PAPER.md:201 (pool member "small MLP ensemble"); Q17: mean of the members' efficiencies */
double kso_ensemble_e(const kso_head *members, int k, const double *x) {
  double sum = 0.0;
  for (int m = 0; m < k; ++m) sum += kso_sigmoid(kso_mlp_z(&members[m], x));
  return sum / (double)k;
}

double kso_predict_one_ensemble(const kso_desc *d, const kso_spec *hw, const kso_head *members, int k,
                                kso_roof *rout, double *e_out) {
  if (d->family == KSO_ALLREDUCE) return kso_predict_one(d, hw, KSO_TIER_NONE, NULL, NULL, rout, e_out);
  kso_roof r;
  kso_roofline(d, hw, &r);
  double x[32];
  kso_features(d, hw, &r, members[0].n_in, x);
  for (int i = 0; i < members[0].n_in; ++i) x[i] = kso_bf16(x[i]);   /* bf16 inputs, Q11 */
  double e = kso_ensemble_e(members, k, x);
  e = dmax(e, ldexp(1.0, -10));                                      /* guard, Q3 */
  if (rout) *rout = r;
  if (e_out) *e_out = e;
  return dmax(r.t_roof / e, hw->t0);
}

int kso_predict_batch_ensemble(int family, int64_t n, const double *const *cols, int n_cols, int64_t s,
                               int64_t hq, int64_t hkv, int64_t dh, const kso_spec *specs, int n_specs,
                               const kso_head *members, int k, double *lat, int64_t *tiles, int64_t *waves,
                               double *troof) {
  if (n < 0 || n_cols < 0 || n_cols > KSO_MAX_COLS || !members || k < 1) return -1;
  for (int m = 1; m < k; ++m) if (members[m].n_in != members[0].n_in) return -1;
  for (int sp = 0; sp < n_specs; ++sp) {
    for (int64_t i = 0; i < n; ++i) {
      kso_desc d;
      d.family = family; d.s = s; d.hq = hq; d.hkv = hkv; d.d = dh;
      for (int c = 0; c < KSO_MAX_COLS; ++c) d.v[c] = (c < n_cols) ? (int64_t)llround(cols[c][i]) : 0;
      kso_roof r;
      const double t = kso_predict_one_ensemble(&d, &specs[sp], members, k, &r, NULL);
      const size_t o = (size_t)sp * (size_t)n + (size_t)i;
      lat[o] = t;
      if (tiles) tiles[o] = r.B;
      if (waves) waves[o] = r.W;
      if (troof) troof[o] = r.t_roof;
    }
  }
  return 0;
}

/* PAPER.md:211 density routing; Q16 */
int kso_in_hull(const kso_grid *g, const kso_desc *d) {
  double v[3];
  kso_grid_axes(d, v);
  for (int a = 0; a < 3; ++a) {
    if (g->dims[a] <= 1) continue;                      /* a flat axis measures nothing: no constraint */
    if (!(v[a] > 0.0)) return 0;
    const double vmin = ceil(exp2(g->lo[a])), vmax = floor(exp2(g->hi[a]));
    if (v[a] < vmin || v[a] > vmax) return 0;
  }
  return 1;
}

double kso_predict_one_routed(const kso_desc *d, const kso_spec *hw, const kso_grid *g, const kso_head *h,
                              const kso_bounded *bh, kso_roof *r, double *e_out, int *routed_out) {
  if (d->family == KSO_ALLREDUCE || kso_in_hull(g, d)) {
    if (routed_out) *routed_out = 0;
    return kso_predict_one(d, hw, KSO_TIER_B, NULL, g, r, e_out);
  }
  if (routed_out) *routed_out = 1;
  if (h) return kso_predict_one(d, hw, KSO_TIER_A, h, NULL, r, e_out);
  return kso_predict_one_bounded(d, hw, bh, r, e_out);
}

int kso_predict_batch_routed(int family, int64_t n, const double *const *cols, int n_cols, int64_t s,
                             int64_t hq, int64_t hkv, int64_t dh, const kso_spec *specs, int n_specs,
                             const kso_grid *g, const kso_head *h, const kso_bounded *bh, double *lat,
                             int64_t *tiles, int64_t *waves, double *troof, int64_t *routed) {
  if (n < 0 || n_cols < 0 || n_cols > KSO_MAX_COLS) return -1;
  if (family != KSO_ALLREDUCE && (!g || (!h && !bh))) return -1;
  for (int sp = 0; sp < n_specs; ++sp) {
    for (int64_t i = 0; i < n; ++i) {
      kso_desc d;
      d.family = family; d.s = s; d.hq = hq; d.hkv = hkv; d.d = dh;
      for (int c = 0; c < KSO_MAX_COLS; ++c) d.v[c] = (c < n_cols) ? (int64_t)llround(cols[c][i]) : 0;
      kso_roof r;
      int fell = 0;
      const double t = kso_predict_one_routed(&d, &specs[sp], g, h, bh, &r, NULL, &fell);
      const size_t o = (size_t)sp * (size_t)n + (size_t)i;
      lat[o] = t;
      if (tiles) tiles[o] = r.B;
      if (waves) waves[o] = r.W;
      if (troof) troof[o] = r.t_roof;
      if (routed && sp == 0) routed[i] = fell;
    }
  }
  return 0;
}

int kso_predict_batch(int family, int64_t n, const double *const *cols, int n_cols, int64_t s,
                      int64_t hq, int64_t hkv, int64_t dh, const kso_spec *specs, int n_specs,
                      int tier, const kso_head *h, const kso_grid *g, double *lat, int64_t *tiles,
                      int64_t *waves, double *troof) {
  if (n < 0 || n_cols < 0 || n_cols > KSO_MAX_COLS) return -1;
  if (tier == KSO_TIER_A && !h && family != KSO_ALLREDUCE) return -1;
  if (tier == KSO_TIER_B && !g && family != KSO_ALLREDUCE) return -1;
  for (int sp = 0; sp < n_specs; ++sp) {
    for (int64_t i = 0; i < n; ++i) {
      kso_desc d;
      d.family = family; d.s = s; d.hq = hq; d.hkv = hkv; d.d = dh;
      for (int c = 0; c < KSO_MAX_COLS; ++c) d.v[c] = (c < n_cols) ? (int64_t)llround(cols[c][i]) : 0;
      kso_roof r;
      double t = kso_predict_one(&d, &specs[sp], tier, h, g, &r, NULL);
      size_t o = (size_t)sp * (size_t)n + (size_t)i;
      lat[o] = t;
      if (tiles) tiles[o] = r.B;
      if (waves) waves[o] = r.W;
      if (troof) troof[o] = r.t_roof;
    }
  }
  return 0;
}

/* ---------------------------------------------------------------- S6 + S7
 * the GPU body of a step is the sum of its kernels' latencies;
 * PAPER.md:233 Eq. 4: t_step = max(t_gpu + n c_disp, l) + max(0, c_ovl - t_gpu) + c_tail. */
void kso_compose(int n_buckets, const double *const *lat, const int64_t *const *step_off,
                 int64_t n_steps, const kso_step_params *p, const int64_t *cfg_off, int64_t n_cfg,
                 double *step_lat, double *cfg_lat) {
  for (int64_t s = 0; s < n_steps; ++s) {
    double sum = 0.0;
    int64_t cnt = 0;
    for (int b = 0; b < n_buckets; ++b) {
      for (int64_t k = step_off[b][s]; k < step_off[b][s + 1]; ++k) { sum += lat[b][k]; cnt += 1; }
    }
    double t_gpu = p->body_scale * sum;
    step_lat[s] = dmax(t_gpu + (double)cnt * p->c_disp, p->floor_l) + dmax(0.0, p->c_ovl - t_gpu) + p->c_tail;
  }
  for (int64_t c = 0; c < n_cfg; ++c) {
    double tot = 0.0;
    for (int64_t s = cfg_off[c]; s < cfg_off[c + 1]; ++s) tot += step_lat[s];
    cfg_lat[c] = tot;
  }
}

/* PAPER.md:231, layer-homogeneous aggregation */
void kso_compose_weighted(int n_buckets, const double *const *lat, const int64_t *const *mult,
                          const int64_t *const *step_off, int64_t n_steps, const kso_step_params *p,
                          const int64_t *cfg_off, int64_t n_cfg, double *step_lat, double *cfg_lat) {
  for (int64_t s = 0; s < n_steps; ++s) {
    double sum = 0.0;
    int64_t cnt = 0;
    for (int b = 0; b < n_buckets; ++b) {
      for (int64_t k = step_off[b][s]; k < step_off[b][s + 1]; ++k) {
        const int64_t m = (mult && mult[b]) ? mult[b][k] : 1;
        sum += (double)m * lat[b][k];
        cnt += m;
      }
    }
    double t_gpu = p->body_scale * sum;
    step_lat[s] = dmax(t_gpu + (double)cnt * p->c_disp, p->floor_l) + dmax(0.0, p->c_ovl - t_gpu) + p->c_tail;
  }
  for (int64_t c = 0; c < n_cfg; ++c) {
    double tot = 0.0;
    for (int64_t s = cfg_off[c]; s < cfg_off[c + 1]; ++s) tot += step_lat[s];
    cfg_lat[c] = tot;
  }
}
