/*
 * fomoe.h — C ABI of the B200-native skip-token MoE layer (FoMoE, arxiv/paper_2606_19025).
 *
 * The library implements the data-parallel hot path of a FoMoE worker's local training step: the
 * partially resident MoE expert layer with the paper's "skip-token" rule, forward and backward, plus
 * the kernel that packs resident-expert parameter deltas for the round-boundary sync.
 *
 * Citations are /root/reference/PAPER.md line numbers (section / equation).
 *
 * General conventions (every entry point):
 *   - Pointers are DEVICE pointers unless the parameter is documented as "host".  The `cfg` structs and
 *     `fomoe_route_state` themselves live on the host; the pointers inside them are device pointers.
 *   - Every buffer is caller-owned.  The library never allocates device memory, frees or keeps a pointer after return.
 *     (Its only own state: one internal non-blocking stream and two events per (host thread, device), created on first use by
 *     fomoe_moe_bwd, which forks the router's backward onto it and joins before returning work to `stream`; the fork /
 *     join are event dependencies, so a step stays capturable in a CUDA graph.  FOMOE_SIDE_STREAM=0 disables it.)
 *     Workspace sizes come from fomoe_workspace_bytes().  All device pointers must be 16-byte aligned.
 *   - Tensors are dense row-major.  Weights are [out,in].  Expert weights are stored ONLY for resident
 *     experts ("the per-worker memory footprint for expert weights decreases") and are
 *     indexed by resident slot: slot i <-> resident_ids[i].
 *   - All work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = default stream).  No entry
 *     point synchronises the device or copies device->host: the number of kept pairs P is never known to
 *     the host, all data-dependent sizes are consumed on the device.
 *   - Return value: FOMOE_OK (0) or a negative error.  Nothing throws across the ABI.  There is NO CPU
 *     fallback: a shape the kernels do not cover returns FOMOE_ERR_UNSUPPORTED.
 *   - dtype: FOMOE_BF16 runs the expert GEMMs on tcgen05 tensor cores (bf16 in, fp32 accumulate in TMEM)
 *     when d_model % 64 == 0 and d_ff % 64 == 0 (otherwise, and for FOMOE_F32, fp32 SIMT kernels).
 *     Router precision (BASELINE.json config 2 "fp32 router"): logits accumulate in fp32.  The fp32 kernels multiply in fp32.
 *     The bf16 tensor-core router (bf16 x, d_model % 64 == 0, E <= 128) multiplies the bf16-exact x with W_r SPLIT into bf16
 *     pieces (hi + mid + lo, each the bf16 rounding of the running residual): 3 pieces = 24 mantissa bits of W_r for E <= 80,
 *     2 pieces = 16 bits for 80 < E <= 128; every product is exact in fp32, the sums are fp32.  Logit error against the fp32
 *     definition: <= ~2e-6 (3 pieces) / <= ~1.6e-5 (2 pieces, d = 4096, |x| ~ 1, |W_r| ~ 0.02): below the 1e-4 margin at which
 *     routing indices are specified to be bit-exact.  The router BACKWARD of the bf16 path runs on bf16 operands (dz, W_r and x
 *     rounded to bf16, fp32 accumulation): dw_router and the router's share of dx carry bf16-level relative error (~4e-3), like
 *     every other gradient of that path.
 */
#ifndef FOMOE_H_
#define FOMOE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FOMOE_ABI_VERSION 5

#if defined(__GNUC__)
#define FOMOE_API __attribute__((visibility("default")))
#else
#define FOMOE_API
#endif

/* status codes */
#define FOMOE_OK 0
#define FOMOE_ERR_BADARG (-1)      /* NULL pointer, non-positive dim, top_k > E, n_res > E, misaligned pointer */
#define FOMOE_ERR_UNSUPPORTED (-2) /* shape outside what the kernels cover (see fomoe_workspace_bytes) */
#define FOMOE_ERR_CUDA (-3)        /* CUDA launch / API failure; text via fomoe_last_cuda_error() */

/* fomoe_config.dtype: element type of x, expert weights, y, dy, dx and expert weight gradients */
#define FOMOE_F32 0
#define FOMOE_BF16 1

/* fomoe_config.gate_fn */
#define FOMOE_GATE_SOFTMAX 0 /* BASELINE.json: softmax over all E logits */
#define FOMOE_GATE_SIGMOID 1 /* paper: independent sigmoid scores, PAPER.md:517 (Eq. 13), 595 (Eq. 17) */

/* fomoe_config.gate_rule: what happens to the gates of surviving pairs when a selected expert is a ghost */
#define FOMOE_DROP_ONLY 0       /* paper: survivors unchanged, skipped pairs contribute 0 */
#define FOMOE_RENORM_TOPK 1     /* g = p / sum over all k selected (resident or not) */
#define FOMOE_RENORM_RESIDENT 2 /* g = p / sum over the kept (resident) selected experts */

/* fomoe_config.expert_fn: form of an expert (routed and shared alike) */
#define FOMOE_EXPERT_SWIGLU 0 /* BASELINE.json: E(x) = W_down (silu(W_gate x) * W_up x), three matrices */
#define FOMOE_EXPERT_SILU 1   /* paper: E(x) = W_down silu(W_up x), "after each expert projection from d_model to d_expert,
                                 the Silu nonlinearity is applied" (§B.3.1); the expert's payload "includes up and
                                 down projection".  W_gate / dW_gate arguments are ignored and may be NULL. */

/* fomoe_config.route_mode */
#define FOMOE_ROUTE_SKIP_TOKEN 0   /* router over all E experts, top-k, THEN ghost pairs are dropped (§3.3.3) */
#define FOMOE_ROUTE_FORCED_LOCAL 1 /* the paper's default mode: the router is partitioned with the experts, "so that individual
                                      tokens are not routed to experts that are unavailable to the local worker"; it
                                      scores only the N_le resident experts (655-660 Eq. 19) and routing is bounded by
                                      min(k, N_le): top_k must be <= n_res.  w_router / dw_router keep the full
                                      [d,E] layout; ghost columns are not read into the decision (their logit is -inf, probability
                                      0) and get zero gradient.  Every selected pair is kept. */

typedef struct fomoe_config {
  int32_t T;           /* tokens (batch x sequence, flattened) */
  int32_t d_model;     /* d */
  int32_t E;           /* routed experts N_e (router width), 1..512 */
  int32_t top_k;       /* k, 1..min(E,32) */
  int32_t d_ff;        /* F: hidden size of a routed expert (d_expert in the paper) */
  int32_t n_shared;    /* always-resident shared experts, 0 if none */
  int32_t d_ff_shared; /* hidden size of a shared expert, 0 if none */
  int32_t dtype;       /* FOMOE_F32 | FOMOE_BF16 */
  int32_t gate_fn;     /* FOMOE_GATE_* */
  int32_t gate_rule;   /* FOMOE_DROP_ONLY | FOMOE_RENORM_* */
  float temperature;   /* tau: logits = x W_r / tau + bias (PAPER.md:175 names it, gives no formula); 1 by default */
  int32_t expert_fn;   /* FOMOE_EXPERT_SWIGLU | FOMOE_EXPERT_SILU */
  int32_t route_mode;  /* FOMOE_ROUTE_SKIP_TOKEN | FOMOE_ROUTE_FORCED_LOCAL */
} fomoe_config;

/*
 * Output of fomoe_route, input of fomoe_moe_fwd / fomoe_moe_bwd.  All pointers: device, caller-owned.
 * P = number of kept (token, expert) pairs = sum_t |topk(t) ∩ S| lives only on the device (offsets[n_res]).
 */
typedef struct fomoe_route_state {
  int32_t* topk_idx;  /* [T,k]  global expert ids, descending logit, ties -> lower id   (Eq. 14) */
  float* gate;        /* [T,k]  gate weight g_tj after the gate rule; exactly 0 for skipped pairs             */
  float* probs;       /* [T,E]  gate-function output p over all E experts (saved for backward)               */
  int32_t* counts;    /* [n_res]    kept pairs per resident slot                                              */
  int32_t* offsets;   /* [n_res+1]  exclusive scan of counts; offsets[n_res] = P                              */
  int32_t* row_token; /* [T*k]  token of row r (rows slot-major, (t,j)-ascending inside a slot); r >= P: -1   */
  int32_t* pair_row;  /* [T,k]  row of pair (t,j), or -1 if its expert is a ghost (skipped)     */
  void* internal;     /* opaque, fomoe_workspace_bytes(...route_internal) bytes: tile-padded row layout       */
} fomoe_route_state;

/*
 * Sizes (bytes) of the three caller-allocated workspaces for (cfg, n_res):
 *   route_internal : fomoe_route_state.internal
 *   saved_acts     : written by fomoe_moe_fwd, read by fomoe_moe_bwd (per padded row: the gathered x row, h, o and the two
 *                    factors the SwiGLU backward multiplies dh with); opaque to the caller
 *   scratch        : temporary inside one fwd or bwd call (may be shared by both, and across layers)
 * Sizes are worst case (every pair kept): rows = T*k + 127*n_res, rounded up to 128.
 * Any out pointer may be NULL.  Returns FOMOE_ERR_BADARG / FOMOE_ERR_UNSUPPORTED for a config the library rejects.
 */
FOMOE_API int fomoe_workspace_bytes(const fomoe_config* cfg, int32_t n_res, size_t* route_internal, size_t* saved_acts,
                          size_t* scratch);

/*
 * Router + gate + top-k + residency mask + permutation  (rows F1-F5 of SURVEY.md §8(a)).
 *   z = x W_r / tau + bias over ALL E experts: the router is not partitioned (Eq. 17);
 *   p = softmax(z) | sigmoid(z);  topk(t) = k largest z;  pair (t,j) kept iff topk_idx[t,j] in S;
 *   gate per cfg->gate_rule;  kept pairs are permuted into per-slot groups (histogram + scan + stable scatter);
 *   skipped pairs get no row.
 * x            [T,d]  cfg->dtype
 * w_router     [d,E]  fp32
 * router_bias  [E] fp32 or NULL (load-skew device of BASELINE.json config 4; gets no gradient)
 * resident_ids [n_res] int32 device, strictly ascending global ids in [0,E).  CONTENT is not validated
 *              (that would need a device sync).  n_res = 0 is legal.
 * out          all arrays written; row_token entries >= P are -1.
 */
FOMOE_API int fomoe_route(const fomoe_config* cfg, const void* x, const float* w_router, const float* router_bias,
                const int32_t* resident_ids, int32_t n_res, const fomoe_route_state* out, void* stream);

/*
 * Forward (rows F6-F8): y_t = sum_{j kept} g_tj W_down,e (silu(W_gate,e x_t) ⊙ W_up,e x_t) + sum_s FFN_s(x_t)
 *   (Eq. 13 over T(x) ∩ S; expert PAPER.md:589 in BASELINE.json's SwiGLU form; shared PAPER.md:86).
 *   Tokens with no kept pair and no shared expert get y_t = 0 exactly.
 *   With cfg->expert_fn == FOMOE_EXPERT_SILU every expert is W_down silu(W_up x) and the *_gate arguments are ignored.
 * w_gate, w_up [n_res,F,d]; w_down [n_res,d,F]  (cfg->dtype; may be NULL iff n_res == 0)
 * sh_gate, sh_up [n_shared,F_sh,d]; sh_down [n_shared,d,F_sh]  (NULL iff n_shared == 0)
 * y [T,d] cfg->dtype, overwritten.   saved_acts, scratch: see fomoe_workspace_bytes.
 */
FOMOE_API int fomoe_moe_fwd(const fomoe_config* cfg, const void* x, const fomoe_route_state* route, int32_t n_res,
                  const void* w_gate, const void* w_up, const void* w_down,
                  const void* sh_gate, const void* sh_up, const void* sh_down,
                  void* y, void* saved_acts, void* scratch, void* stream);

/*
 * Backward (rows B1-B7) for upstream dy [T,d]: gradients of the LOCAL graph only — ghost paths are absent from it
 * and there is no storage for ghost-expert gradients ("each worker responsible solely for updating
 * its local experts").  Must follow fomoe_moe_fwd with the same route and saved_acts.
 * Outputs are OVERWRITTEN (not accumulated):
 *   dx [T,d] cfg->dtype;  dw_router [d,E] fp32 (dense: the router is a dense parameter in skip-token mode);
 *   dw_gate, dw_up [n_res,F,d], dw_down [n_res,d,F] cfg->dtype;  d_sh_* like their weights (NULL iff n_shared == 0).
 */
FOMOE_API int fomoe_moe_bwd(const fomoe_config* cfg, const void* dy, const void* x, const fomoe_route_state* route, int32_t n_res,
                  const float* w_router, const void* w_gate, const void* w_up, const void* w_down,
                  const void* sh_gate, const void* sh_up, const void* sh_down, const void* saved_acts,
                  void* dx, float* dw_router, void* dw_gate, void* dw_up, void* dw_down,
                  void* d_sh_gate, void* d_sh_up, void* d_sh_down, void* scratch, void* stream);

/*
 * Resident-delta pack (row S1): the worker's contribution to the per-expert replica-group all-reduce at a round
 * boundary (Alg. 2 l.19).  For the b-th packed slot s = pack_slots[b] (or b if NULL):
 *   payload[b*block + 0 ..)            = w_start_gate[s] - w_now_gate[s]     (elems_gate words)
 *   payload[b*block + elems_gate ..)   = w_start_up[s]   - w_now_up[s]       (elems_up words)
 *   payload[b*block + elems_gate+elems_up ..) = w_start_down[s] - w_now_down[s]  (elems_down words)
 * block = elems_gate + elems_up + elems_down; an expert's payload is its projections, the router column is excluded
 * in skip-token mode.  All fp32; each word is one IEEE subtraction (bit-exact vs the oracle).
 * w_now / w_start: host arrays of 3 device pointers (gate, up, down), each [n_res, elems_*] fp32.
 * pack_slots: [n_pack] int32 device or NULL (= all slots, n_pack must equal n_res).  elems_* must be multiples of 4.
 * A tensor with elems_* == 0 may be NULL: the paper's two-matrix expert packs up | down only (elems_gate = 0).
 */
FOMOE_API int fomoe_pack_resident_deltas(const float* const w_now[3], const float* const w_start[3], int32_t n_res,
                               int64_t elems_gate, int64_t elems_up, int64_t elems_down,
                               const int32_t* pack_slots, int32_t n_pack, float* payload, void* stream);

/*
 * Peripheral LayerNorm either side of the MoE block:  x_{l+1} = x_l + alpha LN(F(LN(x_l)))
 * (Eq. 15, "normalization exclusively to the residual branches"; depth multiplier alpha on the block
 * output, Fig. 12).  The paper gives no LN formula: standard LayerNorm over d_model with gain, bias and eps
 * (R14).  x, residual, out, dout, dresidual, dx: [T,d_model] in `dtype`; gamma, beta, dgamma, dbeta: fp32 [d_model];
 * stats: fp32 [T,2] = (mean, 1/sqrt(var + eps)) of each row, written by the forward and read by the backward.
 *   fomoe_periln_fwd:  out = (residual ? residual : 0) + alpha (gamma xhat + beta)
 *       pre-LN:  fomoe_periln_fwd(x, g1, b1, residual = NULL, alpha = 1) -> the tokens fomoe_route / fomoe_moe_fwd consume
 *       post-LN: fomoe_periln_fwd(y, g2, b2, residual = x, alpha)        -> x_{l+1}
 *   fomoe_periln_bwd:  dx = (dresidual ? dresidual : 0) + d/dx of alpha (gamma xhat + beta) contracted with dout;
 *                      dgamma, dbeta overwritten (fixed-order reduction: run-to-run identical)
 *       post-LN: fomoe_periln_bwd(dout, y, stats2, g2, alpha, dresidual = NULL) -> dy, the dy of fomoe_moe_bwd
 *       pre-LN:  fomoe_periln_bwd(dxn, x, stats1, g1, 1, dresidual = dout)      -> dx of the whole block (residual path added)
 * partials: device workspace of fomoe_periln_workspace_bytes(T, d_model) bytes.  d_model <= 12800.
 */
FOMOE_API int fomoe_periln_workspace_bytes(int32_t T, int32_t d_model, size_t* partials);
FOMOE_API int fomoe_periln_fwd(int32_t T, int32_t d_model, int32_t dtype, const void* x, const float* gamma, const float* beta, float eps,
                     const void* residual, float alpha, void* out, float* stats, void* stream);
FOMOE_API int fomoe_periln_bwd(int32_t T, int32_t d_model, int32_t dtype, const void* dout, const void* x, const float* stats,
                     const float* gamma, float alpha, const void* dresidual, void* dx, float* dgamma, float* dbeta, float* partials,
                     void* stream);

/*
 * fomoe_periln_bwd without a caller-owned workspace, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid allocation): the per-CTA dgamma / dbeta partial sums live in a static device
 * array of fomoe_periln_bwd_noalloc_max_floats() = 4 Mi floats (16 MiB), which every GPU that loads the library holds until
 * the process exits.  Same arguments (all device pointers, caller-owned), same kernels and the same fixed-order reduction as
 * fomoe_periln_bwd: bit-identical results.  The call allocates nothing (no cudaMalloc / cudaFree / allocating library
 * routine); its only set-up is one cudaGetSymbolAddress per device.
 *   Limit: 2 * min(T, 4 * SM count) * d_model <= 4 Mi (on a 148-SM B200: every T up to d_model = 3543, wider rows only for
 *   fewer tokens).  Beyond it: FOMOE_ERR_UNSUPPORTED, text via fomoe_last_cuda_error(); use fomoe_periln_bwd then.
 *   Sharing: every call on a device uses the same array.  Calls on ONE stream are ordered and safe; calls that overlap on the
 *   GPU (several streams, concurrent graph launches) race on it.  Nothing in it needs clearing between calls (each call
 *   overwrites what it later reads).
 */
FOMOE_API size_t fomoe_periln_bwd_noalloc_max_floats(void);
FOMOE_API int fomoe_periln_bwd_noalloc(int32_t T, int32_t d_model, int32_t dtype, const void* dout, const void* x, const float* stats,
                     const float* gamma, float alpha, const void* dresidual, void* dx, float* dgamma, float* dbeta, void* stream);

/*
 * The same block with the LayerNorms FUSED into the layer's own row kernels ("post-LN + depth multiplier +
 * residual fused into combine"; Eq. 15, 601):
 *   fomoe_moe_fwd_periln = fomoe_moe_fwd, whose combine also writes  out = residual + alpha LN(y)  and stats (y is still written: the
 *       post-LN backward reads it).  Bit-identical to fomoe_moe_fwd followed by fomoe_periln_fwd(y, gamma, beta, eps, residual, alpha).
 *   fomoe_moe_bwd_periln = fomoe_moe_bwd, whose final scatter-sum applies the PRE-LN backward to the gradient it has just summed:
 *       dx = dresidual + LN-backward(dxn; x_raw, stats, gamma), dgamma / dbeta overwritten; dxn (the gradient w.r.t. the layer's
 *       input tokens) is never stored.  Bit-identical to fomoe_moe_bwd followed by fomoe_periln_bwd(dxn, x_raw, stats, gamma, 1,
 *       dresidual).  `x` stays the layer's input (the pre-LN OUTPUT); x_raw is the block input the pre-LN normalised.
 * All pointers device, caller-owned; gamma, beta, dgamma, dbeta fp32 [d_model]; stats fp32 [T,2]; partials as for
 * fomoe_periln_bwd.  d_model must fit the register-resident row shape (a multiple of 8 (bf16) / 4 (fp32), <= 8192 (bf16) /
 * 4096 (fp32)): otherwise FOMOE_ERR_UNSUPPORTED and the caller runs the unfused calls.
 */
typedef struct {
  const float* gamma;   /* [d_model] */
  const float* beta;    /* [d_model] */
  float eps;
  float alpha;          /* depth multiplier on the normalised block output */
  const void* residual; /* [T,d_model] block input x_l */
  void* out;            /* [T,d_model] x_{l+1} */
  float* stats;         /* [T,2] (mean, rstd) of y, for the post-LN backward */
} fomoe_periln_post;
typedef struct {
  const void* x_raw;     /* [T,d_model] block input x_l (what the pre-LN normalised) */
  const float* stats;    /* [T,2] written by the pre-LN forward */
  const float* gamma;    /* [d_model] pre-LN gain */
  const void* dresidual; /* [T,d_model] or NULL: gradient arriving through the residual branch */
  float* dgamma;         /* [d_model] out */
  float* dbeta;          /* [d_model] out */
  float* partials;       /* fomoe_periln_workspace_bytes(T, d_model) bytes */
} fomoe_periln_pre_bwd;
FOMOE_API int fomoe_moe_fwd_periln(const fomoe_config* cfg, const void* x, const fomoe_route_state* route, int32_t n_res,
                  const void* w_gate, const void* w_up, const void* w_down,
                  const void* sh_gate, const void* sh_up, const void* sh_down,
                  void* y, void* saved_acts, void* scratch, const fomoe_periln_post* ln, void* stream);
FOMOE_API int fomoe_moe_bwd_periln(const fomoe_config* cfg, const void* dy, const void* x, const fomoe_route_state* route, int32_t n_res,
                  const float* w_router, const void* w_gate, const void* w_up, const void* w_down,
                  const void* sh_gate, const void* sh_up, const void* sh_down, const void* saved_acts,
                  void* dx, float* dw_router, void* dw_gate, void* dw_up, void* dw_down,
                  void* d_sh_gate, void* d_sh_up, void* d_sh_down, void* scratch, const fomoe_periln_pre_bwd* ln, void* stream);

/*
 * Fused local AdamW over the resident experts ("workers execute AdamW locally on their
 * parameter subsets ... workers maintain history only for their own experts"; Table 7: weight decay 0,
 * betas (0.9, 0.95), eps 1e-8).  The paper prints no formula; this is Loshchilov & Hutter's (R13), in fp32:
 *   m = b1 m + (1-b1) g;  v = b2 v + (1-b2) g^2;  w -= lr wd w;  w -= lr (m / (1-b1^step)) / (sqrt(v / (1-b2^step)) + eps)
 * w_master, m, v: host arrays of 3 device pointers (gate, up, down), each fp32 [n_res, elems_*], updated in place.
 * grad: same shapes in `dtype` (FOMOE_F32 | FOMOE_BF16: what fomoe_moe_bwd wrote).  w_compute: NULL, or 3 device pointers
 * (entries may be NULL) receiving w rounded to `dtype` — the copy the GEMMs read.  step counts from 1.
 * A tensor with elems_* == 0 may be NULL (two-matrix expert).  elems_* must be multiples of 4.
 */
FOMOE_API int fomoe_adamw_resident(float* const w_master[3], const void* const grad[3], float* const m[3], float* const v[3],
                         void* const w_compute[3], int32_t dtype, int32_t n_res, int64_t elems_gate, int64_t elems_up,
                         int64_t elems_down, int32_t step, float lr, float beta1, float beta2, float eps, float weight_decay,
                         void* stream);

/*
 * Outer optimizer step on the receiving side of the round boundary (Alg. 2 l.19-20; "DiLoCo/Nesterov uses
 * server learning rate 0.7 and momentum 0.9").  payload_avg has the layout fomoe_pack_resident_deltas writes
 * ([n_pack, elems_gate + elems_up + elems_down], block b <-> slot pack_slots[b]) and holds the replica-group AVERAGE of
 * delta = w_round_start - w_local (the collective that averages it is out of scope: one GPU).  Per element (fp32):
 *   buf = mu buf + delta;   w = w_start - lr (delta + mu buf)
 * and w is written to w_start (the next round's start), w_now (the local master copy) and, if given, w_compute (rounded to
 * `dtype`).  w_start, w_now, momentum: host arrays of 3 device pointers, fp32 [n_res, elems_*].  Slots not packed are untouched.
 */
FOMOE_API int fomoe_outer_nesterov(float* const w_start[3], float* const w_now[3], float* const momentum[3], void* const w_compute[3],
                         int32_t dtype, const float* payload_avg, int32_t n_res, int64_t elems_gate, int64_t elems_up,
                         int64_t elems_down, const int32_t* pack_slots, int32_t n_pack, float lr, float mu, void* stream);

/*
 * One whole step from HOST buffers (the end-to-end path bench.py times): copies x_host and dy_host to the device,
 * runs fomoe_route + fomoe_moe_fwd + fomoe_moe_bwd, copies y and dx back.  x_host, dy_host, y_host, dx_host:
 * HOST pointers, [T,d] cfg->dtype, ideally pinned.  x_dev, dy_dev, y_dev, dx_dev: device staging buffers [T,d].
 * Three engines work side by side: uploads on `copy_stream` (may equal `stream`), kernels on `stream`, downloads on a
 * stream the library owns (per host thread and device).  Inside one call the dy upload overlaps route + forward and the y
 * download overlaps the backward.  ACROSS calls, the library orders every use of a staging buffer after the previous call's
 * use of the same ADDRESS (it keeps one event per address seen; it never dereferences or frees them): a caller that alternates
 * two (x_dev, dy_dev) pairs gets the next step's uploads, this step's kernels and the previous step's dx download running
 * at the same time -- the step is then bound by the slower of PCIe and compute instead of their sum.
 * defer_join = 0: before returning, `stream` is made to wait for the downloads: y_host and dx_host are complete when
 *                 `stream` completes (and consecutive calls do not overlap).
 * defer_join = 1: downloads are left running; call fomoe_moe_step_host_join(stream) (or synchronise the device) before
 *                 reading y_host / dx_host.
 * Everything else as in the three calls above.  Returns after enqueueing.
 */
FOMOE_API int fomoe_moe_step_host(const fomoe_config* cfg, const void* x_host, const void* dy_host, void* y_host, void* dx_host,
                        void* x_dev, void* dy_dev, void* y_dev, void* dx_dev,
                        const float* w_router, const float* router_bias, const int32_t* resident_ids, int32_t n_res,
                        const fomoe_route_state* route,
                        const void* w_gate, const void* w_up, const void* w_down,
                        const void* sh_gate, const void* sh_up, const void* sh_down,
                        float* dw_router, void* dw_gate, void* dw_up, void* dw_down,
                        void* d_sh_gate, void* d_sh_up, void* d_sh_down,
                        void* saved_acts, void* scratch, void* stream, void* copy_stream, int32_t defer_join);
/* Makes `stream` wait for every download this host thread's fomoe_moe_step_host calls have enqueued so far (current device). */
FOMOE_API int fomoe_moe_step_host_join(void* stream);

/*
 * DEBUG: validates the CONTENT of resident_ids ([n_res] int32, device): every id in [0,E), strictly ascending (so no
 * duplicates).  fomoe_route does not check this because checking needs a device->host copy; THIS call synchronises `stream`.
 * Returns FOMOE_ERR_BADARG (text via fomoe_last_cuda_error()) for a set fomoe_route must not be given: an out-of-range id
 * would index the slot map out of bounds.
 */
FOMOE_API int fomoe_debug_validate_resident(const int32_t* resident_ids, int32_t n_res, int32_t E, void* stream);

/*
 * Routing diagnostics from the output of fomoe_route ("routing entropy, load coefficients of variation, and
 * overflow rates"; under imbalance use "the actual frequency of the token assignments to ghost experts against
 * the total number of assignments").  The layer is dropless, so there is no overflow rate; the realised kept / ghost
 * fractions take its place.  Asynchronous on `stream`, no host sync.
 *   load  [E + 2] int32 device workspace; on return load[e] = assignments (t,j) to expert e over ALL E experts
 *   stats [FOMOE_N_STATS] fp32 device:
 *     FOMOE_STAT_KEPT_FRACTION     P / (T k)            (the realised sigma_st of PAPER.md:200 Eq. 2)
 *     FOMOE_STAT_GHOST_FRACTION    1 - P / (T k)
 *     FOMOE_STAT_ZERO_KEPT_TOKENS  fraction of tokens none of whose k experts is resident
 *     FOMOE_STAT_LOAD_CV           std(load) / mean(load) over the E experts (population std)
 *     FOMOE_STAT_ROUTING_ENTROPY   -sum_e f_e ln f_e, f_e = load[e] / (T k)   (nats; ln E when perfectly balanced)
 *     FOMOE_STAT_MAX_LOAD / FOMOE_STAT_MIN_LOAD
 */
#define FOMOE_STAT_KEPT_FRACTION 0
#define FOMOE_STAT_GHOST_FRACTION 1
#define FOMOE_STAT_ZERO_KEPT_TOKENS 2
#define FOMOE_STAT_LOAD_CV 3
#define FOMOE_STAT_ROUTING_ENTROPY 4
#define FOMOE_STAT_MAX_LOAD 5
#define FOMOE_STAT_MIN_LOAD 6
#define FOMOE_N_STATS 8
FOMOE_API int fomoe_routing_stats(const fomoe_config* cfg, const fomoe_route_state* route, int32_t n_res, int32_t* load, float* stats,
                        void* stream);

/* Number of kernels the last call on this thread launched (bench.py's gpu_launches). */
FOMOE_API int fomoe_last_launch_count(void);

/* Text of the last CUDA error seen by this thread ("" if none). Host pointer, valid until the next failing call. */
FOMOE_API const char* fomoe_last_cuda_error(void);

/* FOMOE_ABI_VERSION the library was built with. */
FOMOE_API int fomoe_abi_version(void);

/* Force the fp32-accumulate SIMT kernels even where tcgen05 applies (1) or not (0); returns the previous value.
 * Debug / A-B testing only. */
FOMOE_API int fomoe_set_force_simt(int on);

/*
 * Per-kernel timing for bench.py's roofline figures.  fomoe_profile_enable(1) clears and starts recording on the
 * calling thread: every kernel the library launches is followed by a CUDA event on its stream.  fomoe_profile_collect
 * synchronises the last event and returns the number of kernel records; for i < min(count, cap) it stores the
 * kernel's name (a static string) and the milliseconds since the previous event on the stream.  Recording adds an
 * event per launch, so timed throughput runs keep it off (fomoe_profile_enable(0)).
 */
FOMOE_API int fomoe_profile_enable(int on);
FOMOE_API int fomoe_profile_collect(const char** names, float* ms, int cap);

#ifdef __cplusplus
}
#endif
#endif /* FOMOE_H_ */
