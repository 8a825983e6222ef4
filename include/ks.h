/* ks.h — C ABI of libks: batched per-kernel latency prediction + serving-step composition,
 * the data-parallel hot path of KernelSight-LM (arxiv 2606.28565), on one B200 (sm_100a).
 *
 * Citations are PAPER.md:<line> (the paper text) or DESIGN.md §3 Q<n> (a stated reading where the
 * paper is silent).  Everything here runs in hand-written CUDA kernels; there is no CPU fallback:
 * every call fails with KS_ECUDA if no sm_100 device/context can be used.
 *
 * Model (Eq. 2):   t = max(t_roof * eta, t0),
 *                               t_roof = max(F_comp / P_peak * u, F_mem / BW_peak),
 *   u = ceil(B/S) * S / B  with S = n_sm * ctas_per_sm CTA slots (Fig. 2; Q4),
 *   eta = 1/e, e in (0,1] from a per-family MLP head over dimensionless features (Tier A,
 *   PAPER.md:199-201) or from trilinear interpolation in a measured efficiency grid (Tier B,
 *   PAPER.md:211), or e = 1 (KS_TIER_NONE).
 * Step composition (Eq. 4):
 *   t_gpu = body_scale * sum_k t_k ;  t_step = max(t_gpu + n c_disp, l) + max(0, c_ovl - t_gpu) + c_tail.
 *
 * Conventions
 *  - Ownership: the library owns only what ks_load_* copies and its internal workspace.  Every
 *    descriptor/offset/output buffer is caller-owned and only borrowed for the duration of the call.
 *  - Memory space: each compute call takes a ks_mem_space saying where ALL its array arguments
 *    (columns, offsets, outputs) live.  KS_MEM_DEVICE: device pointers on the ctx device, 16-byte
 *    aligned; work is enqueued on the ctx stream and the call returns without synchronising.
 *    KS_MEM_HOST: host pointers (pinned or pageable); the library copies inputs to its device
 *    workspace, runs the same kernels, copies results back and synchronises the stream before
 *    returning.  Host structs (ks_desc_batch, ks_hw_spec, ks_step_params, pointer arrays) are always
 *    host memory and are read during the call only.
 *  - Errors: every function returns a ks_status; nothing throws or aborts.  Arguments are validated
 *    before anything is enqueued: on KS_EINVAL / KS_ESTATE / KS_EUNSUPPORTED nothing was written.
 *    A CUDA failure returns KS_ECUDA and is sticky until ks_destroy.
 *  - Determinism: no floating-point atomics; identical inputs give bit-identical outputs.
 */
#ifndef KS_H
#define KS_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define KS_API __attribute__((visibility("default")))
#else
#define KS_API
#endif

typedef struct ks_ctx ks_ctx;   /* opaque; owns device copies of heads and grids + workspace */

typedef enum { KS_OK = 0, KS_EINVAL = 1, KS_ENOMEM = 2, KS_ECUDA = 3, KS_ESTATE = 4, KS_EUNSUPPORTED = 5,
               KS_ELIMIT = 6 /* a fixed capacity was exceeded (ks_predict_routed_static) */ } ks_status;
typedef enum { KS_FAM_GEMM = 0, KS_FAM_GROUPED_GEMM = 1, KS_FAM_ATTN = 2, KS_FAM_ELEMWISE = 3, KS_FAM_ALLREDUCE = 4,
               KS_FAM_COUNT = 5 } ks_family;
typedef enum { KS_TIER_NONE = 0, KS_TIER_A = 1, KS_TIER_B = 2, KS_TIER_B_ROUTED = 3 } ks_tier;
/* Efficiency-model slots.  ks_family says how a bucket's rows are DECODED (which columns, which FLOP/byte/tile
 * formulas); the model slot says which learned head / measured grid PRICES them.  The paper learns eta
 * "separately for each kernel family f.  This includes GEMM, the LM head, attention prefill and decode, and the
 * elementwise and memory kernels" (the families of Tables 2 and 4), which
 * is finer than the decode enum: an LM-head bucket decodes as KS_FAM_GEMM and prefill and decode attention both as
 * KS_FAM_ATTN.  A slot is just an index in [0, KS_MAX_MODEL_SLOTS); the names below are a convention.  Slots 0-4
 * coincide with ks_family, so callers that keep one model per decode family use slot = family
 * (ks_desc_batch.model_slot = KS_SLOT_FAMILY). */
typedef enum { KS_SLOT_FAMILY = -1,   /* in ks_desc_batch.model_slot: the slot numbered like the bucket's family */
               KS_SLOT_GEMM = 0, KS_SLOT_GROUPED_GEMM = 1, KS_SLOT_ATTN = 2, KS_SLOT_ELEMWISE = 3, KS_SLOT_ALLREDUCE = 4,
               KS_SLOT_LM_HEAD = 5, KS_SLOT_ATTN_PREFILL = 6, KS_SLOT_ATTN_DECODE = 7, KS_SLOT_RMSNORM = 8,
               KS_SLOT_SILU_MUL = 9, KS_SLOT_ROPE = 10, KS_SLOT_KV_WRITE = 11, KS_SLOT_EMBEDDING = 12,
               KS_SLOT_RESIDUAL_ADD = 13, KS_MAX_MODEL_SLOTS = 16 } ks_model_slot;
/* What an MLP head's scalar output z means (ks_set_head_output). */
typedef enum { KS_HEAD_UTILISATION = 0,   /* e = sigmoid(z), eta = 1 / e (BASELINE.json "sigmoid out"; Q3) */
               KS_HEAD_LOG_ETA = 1        /* z = log eta: eta = exp(max(z, 0)) >= 1 (PAPER.md:193 "eta >= 1", :199 heads
                                             "trained against log eta"; Q21), capped at 2^10 like the guard */
} ks_head_output;
typedef enum { KS_COL_I32 = 0, KS_COL_F32 = 1 } ks_col_dtype;   /* F32 columns must hold exact integers < 2^24 */
typedef enum { KS_MEM_DEVICE = 0, KS_MEM_HOST = 1 } ks_mem_space;

#define KS_MAX_COLS 10      /* grouped GEMM: N, K, m_0..m_7 */
#define KS_MAX_BATCHES 8    /* family buckets per call */
#define KS_N_EXPERTS 8
#define KS_MAX_GRID_NODES 32768   /* a Tier-B grid is staged whole in shared memory (128 KiB fp32) */

/* Hardware-spec vector (peak compute, peak bandwidth, SM count, cache sizes; Table 5
 * PAPER.md:473-487).  tile_*, ctas_per_sm, ew_elems_per_cta parameterise the CTA count B (Q1, Q4);
 * t0 is the launch floor of Eq. 2.  All integer fields must be >= 1. */
typedef struct {
  float peak_flops;        /* FLOP/s for the descriptor dtype */
  float peak_bw;           /* bytes/s */
  int32_t n_sm, ctas_per_sm, tile_m, tile_n, ew_elems_per_cta;
  float l2_bytes;          /* L2 capacity in bytes */
  float t0;                /* launch floor, seconds (>= 0) */
  float ar_alpha0;         /* interconnect: all-reduce startup/synchronisation term, seconds (>= 0) */
  float ar_beta_eff;       /* interconnect: effective bandwidth, bytes/s (> 0); Eq. 3 */
} ks_hw_spec;

/* One family bucket of kernel-instance descriptors in SoA form.
 * Column meaning by family (all values non-negative integers):
 *   KS_FAM_GEMM          cols = {M, N, K}
 *   KS_FAM_GROUPED_GEMM  cols = {N, K, m_0, ..., m_7}   tokens per expert, shared N, K
 *   KS_FAM_ATTN          cols = {batch, q_len, kv_len}  causal, kv_len >= q_len (smaller kv is raised to q);
 *                        attn_hq / attn_hkv / attn_head_dim are per-bucket constants
 *   KS_FAM_ELEMWISE      cols = {n_elements, subop}     subop: 0 RMSNorm, 1 SiLU*Mul, 2 RoPE,
 *                        3 KV-cache write, 4 embedding, 5 residual add (out-of-range is clamped)
 *   KS_FAM_ALLREDUCE     cols = {S_bytes, P}            tensor-parallel ring all-reduce of S bytes over P
 *                        shards: t = ar_alpha0 + 2 (P-1)/P * S / ar_beta_eff (Eq. 3) under
 *                        every tier (no roofline, no eta, no t0 floor; tiles = waves = 0, t_roof = t);
 *                        it enters the step sum like a kernel
 * Each column has n elements of col_dtype; pointers live in the call's ks_mem_space. */
typedef struct {
  int32_t family;          /* ks_family */
  int32_t n;               /* rows; 0 is a legal no-op */
  int32_t col_dtype;       /* ks_col_dtype */
  int32_t dtype_bytes;     /* s: bytes per tensor element of the modelled kernel (1, 2 or 4) */
  int32_t n_cols;          /* columns supplied; must equal the family's count */
  int32_t attn_hq, attn_hkv, attn_head_dim;
  const void *cols[KS_MAX_COLS];
  int32_t model_slot;      /* efficiency model that prices this bucket: KS_SLOT_FAMILY (-1) or a slot in
                              [0, KS_MAX_MODEL_SLOTS).  NOTE: zero-initialised structs name slot 0 (KS_SLOT_GEMM) */
  const int32_t *mult;     /* optional (may be NULL = all ones): per-row multiplicity m_k >= 0, int32 [n], in the
                              call's memory space.  Layer-homogeneous form of PAPER.md:231 (t_gpu = L t_layer +
                              t_lm_head + t_embed): a row stands for m_k identical kernels of its step.  Read by
                              ks_run_steps only (ks_predict_kernels predicts a row once whatever its multiplicity). */
} ks_desc_batch;

/* Host-overlap constants of Eq. 4; body_scale multiplies sum t (Q7). */
typedef struct { float c_disp, floor_l, c_ovl, c_tail, body_scale; } ks_step_params;

/* Create a context on `device`.  `cuda_stream` is a borrowed cudaStream_t (NULL = legacy default
 * stream) on which all work of this context is enqueued.  KS_ECUDA if the device is not sm_100. */
KS_API ks_status ks_create(ks_ctx **out, int device, void *cuda_stream);

/* Load (or replace) the Tier-A efficiency head of model slot `slot` (0 <= slot < KS_MAX_MODEL_SLOTS; a slot holds
 * ONE Tier-A head of any kind and ONE Tier-B grid): MLP n_in -> h1 -> h2 -> 1 with GELU
 * hidden activations and a sigmoid output giving the efficiency e (sizes and
 * activations BASELINE.json; Q3, Q6).  All arrays are HOST fp32 and are copied: W1[n_in][h1],
 * b1[h1], W2[h1][h2], b2[h2], w3[h2].  Weights are rounded to bf16 (RNE) for the tensor-core
 * contraction; biases keep >= 16 significant bits.  The feature vector is fixed by the library
 * (Q2): n_in must be 8, 12 or 32.  Supported hidden sizes: h1 == h2 in {64, 128, 256};
 * anything else returns KS_EUNSUPPORTED. */
KS_API ks_status ks_load_heads(ks_ctx *ctx, int slot, int n_in, int h1, int h2, const float *W1,
                        const float *b1, const float *W2, const float *b2, const float *w3, float b3);

/* Load (or replace) the Tier-A head of `slot` with an MLP ENSEMBLE ("small MLP ensemble";
 * DESIGN.md Q17): n_members MLPs n_in -> h -> h -> 1 of one shape, each as in ks_load_heads; the efficiency is
 * the arithmetic mean of the members' sigmoid outputs, e = (1/k) sum_m sigmoid(z_m(x)), then the guard and
 * eta = 1/e.  Arrays are HOST fp32 with the member index leading, copied: W1[k][n_in][h], b1[k][h],
 * W2[k][h][h], b2[k][h], w3[k][h], b3[k].  The members run side by side in ONE pass of the Tier-A kernel
 * (layer 1 concatenated, layer 2 block-diagonal), so k * h must be a supported hidden size:
 * h in {32, 64, 128}, k <= KS_MAX_ENSEMBLE, k * h in {64, 128, 256}; anything else KS_EUNSUPPORTED.
 * Replaces any head the slot held. */
#define KS_MAX_ENSEMBLE 8
KS_API ks_status ks_load_head_ensemble(ks_ctx *ctx, int slot, int n_in, int h, int n_members,
                                const float *W1, const float *b1, const float *W2, const float *b2,
                                const float *w3, const float *b3);

/* Load (or replace) the Tier-A head of `slot` with the BOUNDED ANALYTICAL form (PAPER.md:197 Fig. 6, :201;
 * DESIGN.md Q15): utilisation e = gamma(x) - alpha(x) / W with W the kernel's wave count,
 * gamma(x) = sigmoid(w_gamma . x + b_gamma), alpha(x) = max(0, w_alpha . x + b_alpha), e clamped to
 * [2^-10, 1], eta = 1 / e.  x = the library's dimensionless features (Q2) in fp32; n_in in {8, 12, 32}.
 * w_gamma[n_in], w_alpha[n_in]: HOST fp32, copied.  A slot holds ONE Tier-A head: this call replaces
 * an MLP head loaded with ks_load_heads and vice versa.  Runs in the streaming kernel (no contraction). */
KS_API ks_status ks_load_bounded_head(ks_ctx *ctx, int slot, int n_in, const float *w_gamma, float b_gamma,
                               const float *w_alpha, float b_alpha);

/* Load (or replace) the Tier-B measured-efficiency grid of `slot` (Q5).
 * values: HOST fp32 [dims[0]][dims[1]][dims[2]], last index fastest, copied, all finite; each dims[a] >= 1 and
 * the product <= KS_MAX_GRID_NODES.  Axis a spans [lo_log2[a], hi_log2[a]] in log2 units (within [-64, 64]: the
 * axis values are int32) with dims[a] uniformly spaced nodes; queries are clamped to the span.  The axis values
 * are those of the FAMILY of the bucket that uses the slot: GEMM (M, N, K); GROUPED (sum m_e, N, K);
 * ATTN (batch, q_len, kv_len); ELEMWISE (n, 2^subop, 1). */
KS_API ks_status ks_load_grid(ks_ctx *ctx, int slot, const int32_t dims[3], const float lo_log2[3],
                       const float hi_log2[3], const float *values);

/* Say what the scalar output of the MLP head loaded in `slot` means (default after every ks_load_heads:
 * KS_HEAD_UTILISATION).  KS_ESTATE if the slot holds no single MLP head (ensembles and the bounded form have one
 * output convention each: KS_EUNSUPPORTED). */
KS_API ks_status ks_set_head_output(ks_ctx *ctx, int slot, ks_head_output mode);

/* Predict the latency of every (spec, descriptor) pair (steps S1-S5 of DESIGN.md §1).
 *   batches[n_batches]   family buckets (<= KS_MAX_BATCHES)
 *   specs[n_specs]       hardware-spec vectors (host)
 *   tier                 KS_TIER_NONE (e = 1), KS_TIER_A (heads), KS_TIER_B (grids, clamped),
 *                        KS_TIER_B_ROUTED (density routing: the grid inside the measured hull,
 *                        the family's Tier-A head outside it; needs both loaded.  The hull is the grid's
 *                        box, decided on integers: ceil(2^lo_a) <= v_a <= floor(2^hi_a) on every axis with
 *                        more than one node, Q16.  Uses 4 bytes per row of library workspace.)
 *   latency[b]           out, fp32 [n_specs][batches[b].n] seconds
 *   tiles[b], waves[b]   optional out (array pointer or entry may be NULL), int32 [n_specs][n]:
 *                        CTA count B and wave count W = ceil(B/S)
 *   t_roof[b]            optional out, fp32 [n_specs][n]
 * KS_ESTATE if the tier needs a head/grid that was not loaded in a bucket's model slot
 * (KS_FAM_ALLREDUCE buckets need neither). */
KS_API ks_status ks_predict_kernels(ks_ctx *ctx, const ks_desc_batch *batches, int n_batches,
                             const ks_hw_spec *specs, int n_specs, ks_tier tier, ks_mem_space space,
                             float *const *latency, int32_t *const *tiles, int32_t *const *waves,
                             float *const *t_roof);

/* Density-routed prediction that ALLOCATES NOTHING: ks_predict_kernels(..., KS_TIER_B_ROUTED, KS_MEM_DEVICE, ...)
 * for callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it).
 * The routing pass (Q16) needs scratch memory: per bucket, the list of the rows outside the
 * grid's hull and its length.  ks_predict_kernels keeps them in the context's grow-only workspace; this entry point
 * keeps them in ONE fixed array in the library's device image (4 MiB + 4 KiB, held by every GPU that loads libks
 * until the process exits) and calls no cudaMalloc / cudaFree or allocating library routine.
 *   Arguments, layouts, validation and results are those of ks_predict_kernels with tier = KS_TIER_B_ROUTED and
 *   space = KS_MEM_DEVICE (columns and outputs are DEVICE pointers, 16-byte aligned); the same kernels run.
 *   Limit: the rows of all buckets other than KS_FAM_ALLREDUCE (which is never routed) must total at most
 *   KS_STATIC_ROUTE_MAX_ROWS; beyond it the call returns KS_ELIMIT and nothing is enqueued or written.
 *   The array is shared by every context, stream and call on a device and keeps the last call's contents: each
 *   call clears the list lengths it uses (stream-ordered) before its kernels run, so calls in sequence on one
 *   stream are safe; calls that OVERLAP on the GPU (two streams, two contexts on one device) race on it and must be
 *   ordered by the caller.  The first call on a device resolves the array's device address (no allocation). */
#define KS_STATIC_ROUTE_MAX_ROWS (1 << 20)
KS_API ks_status ks_predict_routed_static(ks_ctx *ctx, const ks_desc_batch *batches, int n_batches,
                                          const ks_hw_spec *specs, int n_specs, float *const *latency,
                                          int32_t *const *tiles, int32_t *const *waves, float *const *t_roof);

/* Compose per-kernel latencies into per-step and per-configuration latencies (S6-S7).
 *   latency[b]      fp32 [n_specs][batch_n[b]] as written by ks_predict_kernels
 *   step_off[b]     int32 CSR [n_steps+1]: rows [step_off[b][s], step_off[b][s+1]) of bucket b
 *                   belong to step s (non-decreasing; step_off[b][n_steps] <= batch_n[b])
 *   cfg_off         int32 CSR [n_cfg+1] over steps (may be NULL iff n_cfg == 0)
 *   step_latency    out fp32 [n_specs][n_steps]   (Eq. 4)
 *   cfg_latency     out fp32 [n_specs][n_cfg]     (sum of step latencies, accumulated in fp64) */
KS_API ks_status ks_compose_steps(ks_ctx *ctx, const float *const *latency, const int32_t *const *step_off,
                           const int32_t *batch_n, int n_batches, int n_steps, int n_specs,
                           const ks_step_params *params, const int32_t *cfg_off, int n_cfg,
                           ks_mem_space space, float *step_latency, float *cfg_latency);

/* ks_compose_steps with per-row multiplicities (layer-homogeneous form):
 *   mult[b]   optional int32 [batch_n[b]] (the array pointer or an entry may be NULL = all ones), shared
 *             by all specs: t_gpu = body_scale * sum_k m_k t_k, and Eq. 4's launch count n = sum_k m_k. */
KS_API ks_status ks_compose_steps_weighted(ks_ctx *ctx, const float *const *latency, const int32_t *const *mult,
                                    const int32_t *const *step_off, const int32_t *batch_n, int n_batches,
                                    int n_steps, int n_specs, const ks_step_params *params, const int32_t *cfg_off,
                                    int n_cfg, ks_mem_space space, float *step_latency, float *cfg_latency);

/* Convenience: ks_predict_kernels followed by ks_compose_steps in one call (one pass of the whole
 * hot path; rows with batches[b].mult are weighted as in ks_compose_steps_weighted).  latency may be NULL (or hold NULL entries): per-kernel latencies then stay in the
 * library workspace and only the step/config results are returned.  With KS_MEM_HOST this is the
 * end-to-end call: descriptors and offsets go host->device, results device->host, then sync.  Buckets are
 * pipelined in the caller's order (bucket b is copied while bucket b-1 is predicted: largest first is best);
 * pinned host memory is what makes the copies asynchronous, and the columns of a bucket that lie back to
 * back in host memory (cols[k+1] == cols[k] + 4 n, n a multiple of 4) move with a single copy.
 * KS_MEM_DEVICE with KS_TIER_NONE, one spec vector, int32 columns, at most eight buckets and no grouped-GEMM bucket
 * (config 4a's shape, with or without multiplicities: also what ks_sim_run prices at Tier NONE) runs as ONE kernel plus
 * the totals kernel: the latencies are computed in the
 * step kernel's staging phase instead of being written to HBM and read back, and latency[b] is written only where the
 * caller passed a buffer (none: a step moves the descriptor columns only).  Per-kernel latencies are bit-identical to
 * ks_predict_kernels'; step and configuration latencies are summed in the same fixed order as ks_compose_steps'
 * (bit-identical wherever that call stages a chunk in shared memory, within 2e-6 relative otherwise). */
KS_API ks_status ks_run_steps(ks_ctx *ctx, const ks_desc_batch *batches, const int32_t *const *step_off,
                       int n_batches, const ks_hw_spec *specs, int n_specs, ks_tier tier, int n_steps,
                       const ks_step_params *params, const int32_t *cfg_off, int n_cfg,
                       ks_mem_space space, float *const *latency, float *step_latency, float *cfg_latency);

/* ------------------------------------------------------------------------------------------------
 * Serving scheduler and the closed simulation loop.
 *
 * ks_sched is one replica's scheduler, HOST logic (the paper's scheduler is host code too): "a single
 * token-budget loop advances every request's computed-token count toward its target", with continuous
 * batching, chunked prefill, FCFS queuing and preemption/recompute under KV pressure (
 * the exact rules are DESIGN.md Q18; the two-tier prefix cache of PAPER.md:247 is Q19).  It needs no GPU and no ks_ctx.
 * ks_sim_run closes the loop for many replicas at once: every iteration each unfinished replica forms
 * the batch of its next step, the batches' kernel rows (layer-homogeneous form :231) are
 * priced by ONE pass of the GPU path (ks_run_steps), and each replica's clock advances by its own
 * step time.  All pointers below are HOST pointers. */
typedef struct ks_sched ks_sched;

typedef struct {
  int32_t max_num_batched_tokens;  /* T: token budget of one step, >= 1 */
  int32_t max_num_seqs;            /* most requests running at once, >= 1 */
  int32_t block_size;              /* tokens per KV-cache block, >= 1 */
  int32_t num_blocks;              /* KV-cache blocks, >= 1 */
  int32_t enable_prefix_cache;     /* 0 / 1: content-hashed prefix cache (Q19).  Cached blocks
                                      live in the same num_blocks pool; unreferenced ones are evicted on demand,
                                      least recently released first */
  int32_t disk_blocks;             /* capacity of the persistent disk tier in blocks (LRU); 0 = no disk tier */
} ks_sched_config;

/* Dense decoder the steps are priced for. */
typedef struct {
  int32_t n_layers, hidden, ffn, vocab, hq, hkv, head_dim;
  int32_t dtype_bytes;             /* bytes per tensor element (1, 2 or 4) */
  int32_t tp;                      /* tensor-parallel degree; > 1 adds two all-reduces per layer */
  int32_t fine_slots;              /* 0: every bucket is priced by the model slot of its decode family.  1: the paper's
                                      finer families: the LM-head row gets its own bucket priced by
                                      KS_SLOT_LM_HEAD, prefill chunks (n_new > 1) KS_SLOT_ATTN_PREFILL, decode requests
                                      (n_new = 1) KS_SLOT_ATTN_DECODE; GEMM and elementwise rows keep their family's slot */
} ks_model_desc;

typedef struct {
  int64_t n_steps, tokens_scheduled, n_preemptions;
  int64_t gpu_hit_blocks, disk_hit_blocks, evictions;     /* prefix cache: blocks served by each tier, GPU-tier evictions */
  int32_t n_requests, n_finished, n_running, n_waiting;
  int32_t free_blocks;             /* allocatable blocks: free + cached-but-unreferenced */
  int32_t pad;
} ks_sched_stats;

KS_API ks_status ks_sched_create(ks_sched **out, const ks_sched_config *cfg);
/* Append n requests (arrival time in seconds, prompt tokens >= 1, tokens to emit >= 1).  Queue order is
 * FCFS by (arrival, order of insertion).  KS_EINVAL if a request alone can never fit the KV cache
 * (ceil((prompt + max_new) / block_size) > num_blocks) or a value is not finite / not positive;
 * KS_ESTATE once the first step has been formed. */
KS_API ks_status ks_sched_add_requests(ks_sched *s, int n, const double *arrival, const int32_t *prompt_len,
                                const int32_t *max_new);
/* Same with a shared prefix per request (prefix cache): the first prefix_len[i] prompt tokens of request i are
 * the content named prefix_id[i] >= 0 (0 <= prefix_len <= prompt_len; prefix_id < 0 = no shared prefix).  Two
 * requests with the same prefix_id share their common leading FULL blocks.  Both arrays or neither. */
KS_API ks_status ks_sched_add_prefixed_requests(ks_sched *s, int n, const double *arrival, const int32_t *prompt_len,
                                         const int32_t *max_new, const int32_t *prefix_id, const int32_t *prefix_len);
/* Form the batch of the step that starts at `now`.  Writes up to cap entries (request index, new tokens
 * n_new >= 1, cached history hist = computed tokens before the step) in queue order and their number
 * to *n_sched; KS_EINVAL if cap is too small (max_num_seqs always suffices).  *n_sched == 0 means the
 * replica is idle: *next_arrival then holds the arrival time of the next request, or +inf when every
 * request has finished.  KS_ESTATE if the previous batch has not been committed. */
KS_API ks_status ks_sched_step(ks_sched *s, double now, int32_t cap, int32_t *n_sched, int32_t *req,
                        int32_t *n_new, int32_t *hist, double *next_arrival);
/* The step formed last completes at t_end: computed-token counts advance, requests whose known tokens are
 * all computed emit one token (the first one fixes first_token, the max_new-th finish; the request then
 * leaves and frees its blocks). */
KS_API ks_status ks_sched_commit(ks_sched *s, double t_end);
/* Per-request results, each [n_requests] in insertion order (any pointer may be NULL): time of the first
 * and of the last emitted token (NaN while not reached), number of preemptions, prompt tokens served from
 * the prefix cache over all (re)admissions. */
KS_API ks_status ks_sched_results(ks_sched *s, double *first_token, double *finish, int32_t *n_preempt,
                           int32_t *cached_tokens);
KS_API ks_status ks_sched_get_stats(ks_sched *s, ks_sched_stats *out);
KS_API ks_status ks_sched_destroy(ks_sched *s);

typedef struct {
  int64_t iterations;              /* passes of the GPU path */
  int64_t steps;                   /* serving steps priced, all replicas */
  int64_t rows;                    /* kernel rows priced */
  int64_t kernel_instances;        /* sum of multiplicities = kernel launches those steps stand for */
  double schedule_s, enqueue_s, wait_s, commit_s;  /* host wall time spent forming + packing batches, enqueueing
                                      the GPU pass, waiting for it, and committing the steps */
} ks_sim_stats;

/* Run n_replicas schedulers in lock step until all have finished or max_iters iterations have run
 * (max_iters <= 0: no limit).  clock[r] (in/out) is replica r's simulated time.  Step times are
 * Eq. 4 wall times in fp32 from the GPU path for `spec`, `tier` (heads/grids as loaded in ctx) and
 * `params`; clocks accumulate in double.  Optional log (may be NULL with log_cap 0): step_replica[i],
 * step_time[i] for the i-th priced step in the order they were committed (iteration-major, replica
 * order within an iteration); *n_logged receives the count (steps beyond log_cap are not logged).
 * Blocking; uses the context's stream. */
KS_API ks_status ks_sim_run(ks_ctx *ctx, ks_sched *const *scheds, double *clock, int n_replicas,
                     const ks_model_desc *model, const ks_hw_spec *spec, ks_tier tier,
                     const ks_step_params *params, int64_t max_iters, int32_t *step_replica, float *step_time,
                     int64_t log_cap, int64_t *n_logged, ks_sim_stats *stats);

/* Counters: number of kernel launches this context has enqueued so far (for gpu_launches). */
KS_API ks_status ks_get_launch_count(ks_ctx *ctx, int64_t *out);

/* Tier-A activation mode: 0 = fp32 tanh-form GELU (default: most accurate and, as measured, also the fastest),
 * 1 = packed bf16x2 tanh-form GELU (half the MUFU work, ~4x the activation rounding error; measured 2-5 % SLOWER
 * on B200 because the packing and the bf16x2 FMAs move the bound to the issue slots). */
KS_API ks_status ks_set_gelu_mode(ks_ctx *ctx, int mode);

/* Free everything the context owns.  NULL is a no-op returning KS_OK. */
KS_API ks_status ks_destroy(ks_ctx *ctx);

KS_API const char *ks_status_string(ks_status s);

#ifdef __cplusplus
}
#endif
#endif
