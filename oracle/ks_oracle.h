/* ks_oracle.h — CPU ORACLE for the KernelSight-LM kernel-latency hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded C in double precision,
 * written from /root/reference/PAPER.md (cited as PAPER.md:<line>) and the
 * readings listed in DESIGN.md §3.  It shares no code, header, table or helper
 * with the CUDA path (paper_2606_28565_b200/csrc, include/ks.h) and may be
 * imported / linked / executed only by tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py.
 *
 * One descriptor at a time, in the paper's order:
 *   F_comp, F_mem, B            (PAPER.md:193 names them; formulas = DESIGN.md Q1)
 *   W, u                        (Fig. 2)
 *   t_roof                      (Eq. 2, right half)
 *   eta = 1/e  from Tier A head or Tier B grid
 *   t = max(t_roof*eta, t0)     (Eq. 2, left half; floor after eta PAPER.md:193)
 *   t_ar (all-reduce rows)      (Eq. 3; enters the step sum like a kernel)
 *   t_gpu = body_scale*sum t
 *   t_step                      (Eq. 4)
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Fig. 2's worked example, hand-computed
 * rooflines (tests/golden/roofline_cases.txt), brute-force wave/tile/pair counts,
 * numpy+scipy MLP, scipy RegularGridInterpolator, torch bf16 rounding, np.add.reduceat,
 * Eq. 4 regimes, the bounded head's closed forms (alpha = 0, constant maps, W -> inf, numpy dot), Eq. 3 special cases (P = 1, P = 2, P -> inf, linearity in S, a hand-computed case).  Parity unpinned: NONE of the functions below — but note the
 * *feature list* (kso_features) is a reading (Q2): its closed-form special
 * cases are pinned, the paper prints no values for it.
 */
#ifndef KS_ORACLE_H
#define KS_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { KSO_GEMM = 0, KSO_GROUPED = 1, KSO_ATTN = 2, KSO_ELEMWISE = 3, KSO_ALLREDUCE = 4 };
enum { KSO_TIER_NONE = 0, KSO_TIER_A = 1, KSO_TIER_B = 2, KSO_TIER_B_ROUTED = 3 };
#define KSO_MAX_COLS 10
#define KSO_EXPERTS 8

typedef struct {           /* hardware-spec vector, PAPER.md:205 (+ tile/CTA fields, BASELINE.json) */
  double peak_flops, peak_bw;
  int64_t n_sm, ctas_per_sm, tile_m, tile_n, ew_elems_per_cta;
  double l2_bytes, t0;
  double ar_alpha0, ar_beta_eff; /* interconnect: all-reduce startup [s] and effective bandwidth [B/s], Eq. 3 */
} kso_spec;

typedef struct {           /* one kernel-instance descriptor */
  int family;
  int64_t v[KSO_MAX_COLS]; /* GEMM M,N,K | GROUPED N,K,m0..m7 | ATTN B,q,kv | ELEMWISE n,subop | ALLREDUCE S,P */
  int64_t s;               /* bytes per element */
  int64_t hq, hkv, d;      /* attention constants */
} kso_desc;

typedef struct {           /* everything Eq. 2's right half produces for one (descriptor, spec) */
  double F, Y;             /* F_comp [FLOP], F_mem [B] */
  int64_t B, W;            /* CTA/tile count, wave count */
  double u, t_comp, t_mem, t_roof;
} kso_roof;

typedef struct {           /* Tier A head: MLP n_in -> h1 -> h2 -> 1 (GELU hidden units) */
  int n_in, h1, h2;
  const double *W1, *b1, *W2, *b2, *w3; /* W1[n_in][h1], W2[h1][h2]; already bf16-rounded weights */
  double b3;
  int log_eta;             /* what the output z means: 0 = utilisation, e = sigmoid(z) (BASELINE.json; Q3);
                              1 = z is log eta ("trained against log eta"): eta = exp(max(z, 0)) >= 1
                              (PAPER.md:193), Q21 */
} kso_head;

typedef struct {           /* Tier B measured-efficiency grid */
  int64_t dims[3];
  double lo[3], hi[3];     /* log2 span per axis */
  const double *values;    /* [d0][d1][d2], last fastest */
} kso_grid;

typedef struct {           /* bounded analytical head, PAPER.md:197 Fig. 6, :201; maps = DESIGN.md Q15 */
  int n_in;
  const double *w_gamma, *w_alpha; /* [n_in] */
  double b_gamma, b_alpha;
} kso_bounded;

typedef struct { double c_disp, floor_l, c_ovl, c_tail, body_scale; } kso_step_params; /* Eq. 4 */

/* round-to-nearest-even to bfloat16 precision (8 significant bits), returned as double */
double kso_bf16(double x);
/* exact GELU 0.5 x (1 + erf(x / sqrt 2)) and logistic sigmoid */
double kso_gelu(double x);
double kso_sigmoid(double z);
/* eta of a head whose output is log eta, floored at the roofline bound eta >= 1 (Q21) */
double kso_eta_from_log(double z);
/* utilisation e = 1 / eta that an MLP head gives for the (bf16-rounded) features x, by its output convention */
double kso_head_e(const kso_head *h, const double *x);

/* Tensor-parallel ring all-reduce, Eq. 3: t_ar = alpha0 + 2 (P - 1) / P * S / beta_eff
 * (S message bytes, P shards; P <= 1 moves nothing: t_ar = alpha0).  No roofline, no eta, no t0 floor. */
double kso_allreduce(int64_t S, int64_t P, const kso_spec *hw);
/* S1: F_comp, F_mem, B for one descriptor (Q1) */
void kso_work(const kso_desc *d, const kso_spec *hw, double *F, double *Y, int64_t *B);
/* causal (query, key) pair count of a q-token chunk over kv cached+own tokens */
int64_t kso_attn_pairs(int64_t q, int64_t kv);
/* S2: wave quantization W = ceil(B/S), u = W S / B; B = 0 -> W = 0, u = 1 */
void kso_wave(int64_t B, int64_t S, int64_t *W, double *u);
/* S1+S2: Eq. 2 right half */
void kso_roofline(const kso_desc *d, const kso_spec *hw, kso_roof *r);
/* S3: dimensionless features x[0..n_in) (Q2), NOT yet bf16-rounded; n_in in {8,12,32} */
void kso_features(const kso_desc *d, const kso_spec *hw, const kso_roof *r, int n_in, double *x);
/* S4a: z = w3 . g(W2^T g(W1^T x + b1) + b2) + b3, scalar triple loop, double accumulation */
double kso_mlp_z(const kso_head *h, const double *x);
/* S4b: trilinear interpolation of the stored efficiency at axis values v[3] (Q5) */
double kso_trilinear(const kso_grid *g, const double v[3]);
/* Tier-B axis values of a descriptor: GEMM (M,N,K); GROUPED (sum m,N,K); ATTN (B,q,kv);
 * ELEMWISE (n, 2^subop, 1) */
void kso_grid_axes(const kso_desc *d, double v[3]);
/* Bounded analytical head: utilisation e = gamma(x) - alpha(x) / W, eta = 1 / e, with
 * gamma(x) = sigmoid(w_gamma . x + b_gamma) in (0,1) and alpha(x) = max(0, w_alpha . x + b_alpha)
 * (Q15); x = the dimensionless features in full precision (no tensor core on this path);
 * e is clamped to [2^-10, 1]; W = 0 (empty kernel) gives e = gamma. */
double kso_bounded_e(const kso_bounded *bh, const double *x, int64_t W);
/* One full prediction with the bounded head: t = max(t_roof / e, t0). */
double kso_predict_one_bounded(const kso_desc *d, const kso_spec *hw, const kso_bounded *bh, kso_roof *r,
                               double *e_out);
int kso_predict_batch_bounded(int family, int64_t n, const double *const *cols, int n_cols, int64_t s,
                              int64_t hq, int64_t hkv, int64_t dh, const kso_spec *specs, int n_specs,
                              const kso_bounded *bh, double *lat, int64_t *tiles, int64_t *waves, double *troof);
/* MLP ensemble ("small MLP ensemble"; Q17): k members of the same shape, each the
 * MLP of kso_mlp_z; the ensemble's efficiency is the arithmetic mean of the members' outputs,
 * e = (1/k) sum_m sigmoid(z_m(x)), taken before the guard and the inversion eta = 1/e. */
double kso_ensemble_e(const kso_head *members, int k, const double *x);
/* One full prediction with an ensemble head: bf16 inputs as for a single MLP head (Q11). */
double kso_predict_one_ensemble(const kso_desc *d, const kso_spec *hw, const kso_head *members, int k,
                                kso_roof *r, double *e_out);
int kso_predict_batch_ensemble(int family, int64_t n, const double *const *cols, int n_cols, int64_t s,
                               int64_t hq, int64_t hkv, int64_t dh, const kso_spec *specs, int n_specs,
                               const kso_head *members, int k, double *lat, int64_t *tiles, int64_t *waves,
                               double *troof);
/* Density routing: 1 iff the query lies inside the measured hull, here the grid's box:
 * lo_a <= log2 v_a <= hi_a on every axis with more than one node, decided on integers as
 * ceil(2^lo_a) <= v_a <= floor(2^hi_a) (Q16); a non-positive axis value is outside. */
int kso_in_hull(const kso_grid *g, const kso_desc *d);
/* Density-routed Tier B: interpolate the grid inside the hull, otherwise fall back to the family's learned
 * Tier-A head (MLP `h`, or the bounded form `bh` when h is NULL).  routed_out (may be NULL): 1 = fell back. */
double kso_predict_one_routed(const kso_desc *d, const kso_spec *hw, const kso_grid *g, const kso_head *h,
                              const kso_bounded *bh, kso_roof *r, double *e_out, int *routed_out);
int kso_predict_batch_routed(int family, int64_t n, const double *const *cols, int n_cols, int64_t s,
                             int64_t hq, int64_t hkv, int64_t dh, const kso_spec *specs, int n_specs,
                             const kso_grid *g, const kso_head *h, const kso_bounded *bh, double *lat,
                             int64_t *tiles, int64_t *waves, double *troof, int64_t *routed);
/* S5: one full prediction. head/grid may be NULL unless the tier needs them.
 * Returns latency; optional outputs via r (may be NULL) and e_out (may be NULL). */
double kso_predict_one(const kso_desc *d, const kso_spec *hw, int tier, const kso_head *h,
                       const kso_grid *g, kso_roof *r, double *e_out);

/* Batch form over SoA columns given as doubles (exact for the integer inputs used).
 * Outputs are [n_specs][n]; tiles/waves/troof may be NULL. Returns 0, or -1 on bad arguments. */
int kso_predict_batch(int family, int64_t n, const double *const *cols, int n_cols, int64_t s,
                      int64_t hq, int64_t hkv, int64_t dh, const kso_spec *specs, int n_specs,
                      int tier, const kso_head *h, const kso_grid *g, double *lat, int64_t *tiles,
                      int64_t *waves, double *troof);

/* S6+S7: t_gpu[s] = body_scale * sum_b sum_{k in seg} lat_b[k]; n[s] = kernel count;
 * Eq. 4; T_cfg = sum of t_step over the config's steps.  Naive loops in double. */
void kso_compose(int n_buckets, const double *const *lat, const int64_t *const *step_off,
                 int64_t n_steps, const kso_step_params *p, const int64_t *cfg_off, int64_t n_cfg,
                 double *step_lat, double *cfg_lat);

/* Layer-homogeneous form of S6 ("since decoder layers are homogeneous, the GPU body of a
 * step is t_gpu = L t_layer + t_lm_head + t_embed"): every descriptor row carries a multiplicity m_k >= 0
 * (how many identical kernels of the step it stands for; mult[b] == NULL means all ones):
 * t_gpu = body_scale * sum_k m_k t_k, and Eq. 4's launch count is n = sum_k m_k. */
void kso_compose_weighted(int n_buckets, const double *const *lat, const int64_t *const *mult,
                          const int64_t *const *step_off, int64_t n_steps, const kso_step_params *p,
                          const int64_t *cfg_off, int64_t n_cfg, double *step_lat, double *cfg_lat);

#ifdef __cplusplus
}
#endif
#endif
