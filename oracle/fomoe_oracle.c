/*
 * ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow CPU statement of what the skip-token, partially resident MoE layer computes
 * (FoMoE, arxiv/paper_2606_19025), written from /root/reference/PAPER.md, per token, in the paper's
 * order.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this.  It shares no code, header, table or helper with the CUDA path and neither imports the
 * other.
 *
 * Compiled twice from this one file: -DREAL=double (liboracle_f64.so: the parity reference and the
 * finite-difference build) and -DREAL=float (liboracle_f32.so: the "plain fp32 CPU implementation"
 * BASELINE.json names, which is what is timed as cpu_baseline).  OpenMP over tokens / experts only;
 * no BLAS, no blocking, no fusion.
 *
 * Notation: T tokens, d = d_model, E routed experts N_e, k = top-k, F = d_ff,
 * S = resident set (ascending global ids resident_ids[n_res]; slot i <-> resident_ids[i]),
 * weights [out,in] row-major: W_gate,W_up [n_res,F,d], W_down [n_res,d,F], router W_r [d,E].
 *
 * Passages followed:
 *   router over ALL experts, unpartitioned ............ PAPER.md:159 (§3.3.3), 595 (Eq. 17)
 *   gate p = sigmoid(z) (paper) | softmax(z) (BASELINE.json) PAPER.md:517 (Eq. 13), 521, 593-595
 *   top-k on the scores ................................ PAPER.md:519 (Eq. 14)
 *   ghost experts: pairs whose expert is not in S are bypassed,
 *     "ignored by the local computational graph" ....... PAPER.md:157-159, 147 (Fig. 3)
 *   no renormalisation over the surviving experts ...... PAPER.md:593 (§B.3.2)
 *   y = sum_{i in T(x) ∩ S} s_i(x) E_i(x) .............. PAPER.md:515 (Eq. 13)
 *   expert = projection -> SiLU -> projection, E(x) = W_down silu(W_up x) (EXPERT_SILU);
 *     BASELINE.json's configs fix the SwiGLU form
 *     E(x) = W_down (silu(W_gate x) ⊙ W_up x) (EXPERT_SWIGLU) PAPER.md:589 (§B.3.1), 253
 *   shared experts: fully replicated dense components .. PAPER.md:86 (§3.2)
 *   delta payload per resident expert (up+down, router
 *     column excluded in skip-token mode) .............. PAPER.md:253, 824 (Alg. 2 l.19)
 * Readings where the paper is silent are DESIGN.md "Readings" R1..R12 (tie-break, temperature, bias,
 * delta sign, renorm variants).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): brute-force per-token Python loops; torch CPU autograd of
 * an independently written dense "all experts, zeroed W_down" MoE; central finite differences (f64);
 * closed forms (E=1 sigmoid; k=E softmax mixture; n_res=0; hand-derived golden example
 * tests/golden/tiny_moe.json); invariants (counts, offsets, inverse maps, zero rows).  The two
 * RENORM rules are pinned by FD + brute force only (weaker; stated in DESIGN.md).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef REAL
#define REAL double
#endif

enum { GATE_SOFTMAX = 0, GATE_SIGMOID = 1 };
enum { RULE_DROP_ONLY = 0, RULE_RENORM_TOPK = 1, RULE_RENORM_RESIDENT = 2 };
/* expert form: SwiGLU (BASELINE.json's five configs) or the paper's own sigma-MoE expert
 * E(x) = W_down SiLU(W_up x): "After each expert projection from d_model to d_expert, the Silu nonlinearity is applied"
 * (§B.3.1); the expert payload "includes up and down projection".  In the SiLU form W_gate does
 * not exist (pointers may be NULL, dw_gate is not written). */
enum { EXPERT_SWIGLU = 0, EXPERT_SILU = 1 };
/* routing mode.  SKIP_TOKEN: the router is not partitioned, top-k over all E, ghost pairs dropped afterwards.
 * FORCED_LOCAL: the paper's default outside §3.3.3 — the router is partitioned along with the experts "so that individual
 * tokens are not routed to experts that are unavailable to the local worker", it "scores only N_le experts"
 * (655-660 Eq. 19) and local routing is bounded by min(k, N_le): the caller passes
 * k <= n_res.  Written out: the logits of non-resident experts do not exist (-inf here, probability 0), gate and top-k run
 * over the resident ones, every selected pair is kept. */
enum { ROUTE_SKIP_TOKEN = 0, ROUTE_FORCED_LOCAL = 1 };

int oracle_real_bytes(void) { return (int)sizeof(REAL); }

static REAL sigmoid_(REAL v) { return (REAL)1 / ((REAL)1 + (REAL)exp(-(double)v)); }

static REAL dot_(const REAL* a, const REAL* b, int n) {
  REAL s = 0;
#pragma omp simd reduction(+ : s)
  for (int i = 0; i < n; ++i) s += a[i] * b[i];
  return s;
}
static void axpy_(REAL alpha, const REAL* x, REAL* y, int n) {
#pragma omp simd
  for (int i = 0; i < n; ++i) y[i] += alpha * x[i];
}

/* slot_of[e] = resident slot of global expert e, or -1 for a ghost expert. */
static int* make_slot_of(int E, const int32_t* resident_ids, int n_res) {
  int* slot_of = (int*)malloc(sizeof(int) * (size_t)(E > 0 ? E : 1));
  for (int e = 0; e < E; ++e) slot_of[e] = -1;
  for (int i = 0; i < n_res; ++i) slot_of[resident_ids[i]] = i;
  return slot_of;
}

/* ------------------------------------------------------------------------------------------------
 * Steps 1-6 of SURVEY.md §8(c): router, gate, top-k, residency mask, gate rule, permutation.
 * Outputs: logits z [T,E]; probs p [T,E]; topk_idx [T,k] (global ids, descending z, ties -> lower id);
 * gate g [T,k] (0 for skipped pairs); counts [n_res]; offsets [n_res+1]; row_token [T*k] (first P
 * valid, rest -1); pair_row [T,k] (row of the pair in slot-major order, or -1 if skipped).
 * ---------------------------------------------------------------------------------------------- */
int oracle_route(int T, int d, int E, int k, int gate_fn, int gate_rule, double tau, int route_mode,
                 const REAL* x, const REAL* w_r, const REAL* bias,
                 const int32_t* resident_ids, int n_res,
                 REAL* logits, REAL* probs, int32_t* topk_idx, REAL* gate,
                 int32_t* counts, int32_t* offsets, int32_t* row_token, int32_t* pair_row) {
  if (T < 0 || d <= 0 || E <= 0 || k <= 0 || k > E || n_res < 0 || n_res > E) return -1;
  if (route_mode == ROUTE_FORCED_LOCAL && k > n_res) return -1; /* bounded by min(k, N_le) */
  int* slot_of = make_slot_of(E, resident_ids, n_res);

#pragma omp parallel for schedule(static)
  for (int t = 0; t < T; ++t) {
    const REAL* xt = x + (size_t)t * d;
    REAL* z = logits + (size_t)t * E;
    REAL* p = probs + (size_t)t * E;
    /* 1. z_te = (sum_i x_ti W_r[i,e]) / tau + b_e, all E experts */
    for (int e = 0; e < E; ++e) {
      REAL s = 0;
      for (int i = 0; i < d; ++i) s += xt[i] * w_r[(size_t)i * E + e];
      z[e] = s / (REAL)tau + (bias ? bias[e] : (REAL)0);
      if (route_mode == ROUTE_FORCED_LOCAL && slot_of[e] < 0) z[e] = (REAL)-INFINITY; /* no router column for it */
    }
    /* 2. gate function (PAPER.md:517 sigmoid; BASELINE.json softmax, max-subtracted) */
    if (gate_fn == GATE_SIGMOID) {
      for (int e = 0; e < E; ++e) p[e] = sigmoid_(z[e]);
    } else {
      REAL m = (REAL)-INFINITY, sum = 0;
      for (int e = 0; e < E; ++e) m = z[e] > m ? z[e] : m;
      for (int e = 0; e < E; ++e) { p[e] = (REAL)exp((double)(z[e] - m)); sum += p[e]; }
      for (int e = 0; e < E; ++e) p[e] /= sum;
    }
    /* 3. top-k: k selection passes; strict '>' keeps the lower index on ties */
    int32_t* idx = topk_idx + (size_t)t * k;
    for (int j = 0; j < k; ++j) {
      int best = -1;
      for (int e = 0; e < E; ++e) {
        int taken = 0;
        for (int jj = 0; jj < j; ++jj) taken |= (idx[jj] == e);
        if (taken) continue;
        if (best < 0 || z[e] > z[best]) best = e;
      }
      idx[j] = best;
    }
    /* 4.-5. residency mask and gate rule (593) */
    REAL* g = gate + (size_t)t * k;
    REAL s_all = 0, s_kept = 0;
    for (int j = 0; j < k; ++j) {
      s_all += p[idx[j]];
      if (slot_of[idx[j]] >= 0) s_kept += p[idx[j]];
    }
    for (int j = 0; j < k; ++j) {
      if (slot_of[idx[j]] < 0) { g[j] = 0; continue; }
      REAL pj = p[idx[j]];
      g[j] = gate_rule == RULE_DROP_ONLY ? pj : gate_rule == RULE_RENORM_TOPK ? pj / s_all : pj / s_kept;
    }
  }

  /* 6. counts, exclusive scan, rows inside a slot in ascending (t, j) */
  for (int i = 0; i < n_res; ++i) counts[i] = 0;
  for (int t = 0; t < T; ++t)
    for (int j = 0; j < k; ++j) {
      int s = slot_of[topk_idx[(size_t)t * k + j]];
      if (s >= 0) counts[s]++;
    }
  offsets[0] = 0;
  for (int i = 0; i < n_res; ++i) offsets[i + 1] = offsets[i] + counts[i];
  int32_t* cursor = (int32_t*)malloc(sizeof(int32_t) * (size_t)(n_res + 1));
  for (int i = 0; i < n_res; ++i) cursor[i] = offsets[i];
  for (size_t r = 0; r < (size_t)T * k; ++r) row_token[r] = -1;
  for (int t = 0; t < T; ++t)
    for (int j = 0; j < k; ++j) {
      int s = slot_of[topk_idx[(size_t)t * k + j]];
      if (s >= 0) {
        int r = cursor[s]++;
        row_token[r] = t;
        pair_row[(size_t)t * k + j] = r;
      } else {
        pair_row[(size_t)t * k + j] = -1;
      }
    }
  free(cursor);
  free(slot_of);
  return 0;
}

/* One expert on one token.
 * SwiGLU: a = W_g x, u = W_u x, h = a*sigmoid(a) ⊙ u, o = W_d h.
 * SiLU: a = W_u x, h = a*sigmoid(a), o = W_d h   (u is set to 1 so the shared backward formulas hold). */
static void expert_fwd_(int expert_fn, const REAL* xt, int d, int F, const REAL* wg, const REAL* wu, const REAL* wd,
                        REAL* a, REAL* u, REAL* h, REAL* o) {
  for (int f = 0; f < F; ++f) {
    if (expert_fn == EXPERT_SILU) {
      a[f] = dot_(wu + (size_t)f * d, xt, d);
      u[f] = (REAL)1;
    } else {
      a[f] = dot_(wg + (size_t)f * d, xt, d);
      u[f] = dot_(wu + (size_t)f * d, xt, d);
    }
    h[f] = a[f] * sigmoid_(a[f]) * u[f];
  }
  if (o)
    for (int i = 0; i < d; ++i) o[i] = dot_(wd + (size_t)i * F, h, F);
}

/* ------------------------------------------------------------------------------------------------
 * Steps 7-8: y_t = sum_{j kept, ascending j} g_tj * E_{e_tj}(x_t) + sum_s FFN_s(x_t)   (86)
 * Tokens with no kept pair and no shared expert give y_t = 0 exactly.
 * ---------------------------------------------------------------------------------------------- */
int oracle_moe_fwd(int T, int d, int E, int k, int F, int n_sh, int F_sh, int expert_fn,
                   const REAL* x, const int32_t* topk_idx, const REAL* gate,
                   const int32_t* resident_ids, int n_res,
                   const REAL* w_gate, const REAL* w_up, const REAL* w_down,
                   const REAL* sh_gate, const REAL* sh_up, const REAL* sh_down,
                   REAL* y) {
  int* slot_of = make_slot_of(E, resident_ids, n_res);
  int Fm = F > F_sh ? F : F_sh;
#pragma omp parallel
  {
    REAL* a = (REAL*)malloc(sizeof(REAL) * (size_t)(3 * Fm + d));
    REAL *u = a + Fm, *h = u + Fm, *o = h + Fm;
#pragma omp for schedule(dynamic, 8)
    for (int t = 0; t < T; ++t) {
      const REAL* xt = x + (size_t)t * d;
      REAL* yt = y + (size_t)t * d;
      for (int i = 0; i < d; ++i) yt[i] = 0;
      for (int j = 0; j < k; ++j) {
        int s = slot_of[topk_idx[(size_t)t * k + j]];
        if (s < 0) continue; /* ghost expert: skipped */
        expert_fwd_(expert_fn, xt, d, F, w_gate ? w_gate + (size_t)s * F * d : NULL, w_up + (size_t)s * F * d, w_down + (size_t)s * d * F, a, u, h, o);
        axpy_(gate[(size_t)t * k + j], o, yt, d);
      }
      for (int s = 0; s < n_sh; ++s) {
        expert_fwd_(expert_fn, xt, d, F_sh, sh_gate ? sh_gate + (size_t)s * F_sh * d : NULL, sh_up + (size_t)s * F_sh * d, sh_down + (size_t)s * d * F_sh, a, u, h, o);
        axpy_((REAL)1, o, yt, d);
      }
    }
    free(a);
  }
  free(slot_of);
  return 0;
}

/* Backward of one expert on one token given do = dL/do.  Adds W_g^T da + W_u^T du into dx_acc (if
 * non-NULL) and the rank-1 weight-gradient terms into dwg/dwu/dwd (if non-NULL). Returns via a,u,h the
 * recomputed forward. */
static void expert_bwd_(int expert_fn, const REAL* xt, const REAL* dov, int d, int F,
                        const REAL* wg, const REAL* wu, const REAL* wd,
                        REAL* a, REAL* u, REAL* h, REAL* dh, REAL* dx_acc,
                        REAL* dwg, REAL* dwu, REAL* dwd) {
  expert_fwd_(expert_fn, xt, d, F, wg, wu, wd, a, u, h, NULL);
  for (int f = 0; f < F; ++f) dh[f] = 0;
  for (int i = 0; i < d; ++i) axpy_(dov[i], wd + (size_t)i * F, dh, F); /* dh = W_d^T do */
  if (dwd)
    for (int i = 0; i < d; ++i) axpy_(dov[i], h, dwd + (size_t)i * F, F); /* dW_d += do h^T */
  for (int f = 0; f < F; ++f) {
    REAL sg = sigmoid_(a[f]);
    REAL da = dh[f] * u[f] * sg * ((REAL)1 + a[f] * ((REAL)1 - sg)); /* d silu(a)/da = sg (1 + a (1 - sg)) */
    REAL du = dh[f] * a[f] * sg;
    if (expert_fn == EXPERT_SILU) { /* a = W_u x is the only projection: da flows into W_up, there is no u path */
      if (dx_acc) axpy_(da, wu + (size_t)f * d, dx_acc, d);
      if (dwu) axpy_(da, xt, dwu + (size_t)f * d, d);
      continue;
    }
    if (dx_acc) {
      axpy_(da, wg + (size_t)f * d, dx_acc, d);
      axpy_(du, wu + (size_t)f * d, dx_acc, d);
    }
    if (dwg) {
      axpy_(da, xt, dwg + (size_t)f * d, d);
      axpy_(du, xt, dwu + (size_t)f * d, d);
    }
  }
}

/* ------------------------------------------------------------------------------------------------
 * Step 9: backward of steps 1-8 for an upstream dy (the local computational graph only).
 * Outputs (all overwritten): dx [T,d]; dw_router [d,E]; dw_gate, dw_up [n_res,F,d]; dw_down [n_res,d,F];
 * d_sh_* like their weights; dgate [T,k] (dL/dg_tj, 0 for skipped pairs); dlogits [T,E].
 * ---------------------------------------------------------------------------------------------- */
int oracle_moe_bwd(int T, int d, int E, int k, int F, int n_sh, int F_sh, int expert_fn,
                   int gate_fn, int gate_rule, double tau,
                   const REAL* x, const REAL* dy, const REAL* w_r,
                   const REAL* probs, const int32_t* topk_idx, const REAL* gate,
                   const int32_t* resident_ids, int n_res,
                   const int32_t* offsets, const int32_t* row_token,
                   const REAL* w_gate, const REAL* w_up, const REAL* w_down,
                   const REAL* sh_gate, const REAL* sh_up, const REAL* sh_down,
                   REAL* dx, REAL* dw_router, REAL* dw_gate, REAL* dw_up, REAL* dw_down,
                   REAL* d_sh_gate, REAL* d_sh_up, REAL* d_sh_down,
                   REAL* dgate, REAL* dlogits) {
  int* slot_of = make_slot_of(E, resident_ids, n_res);
  int Fm = F > F_sh ? F : F_sh;

  /* Phase 1, per token: dgate, dx (expert + shared + router terms), dlogits. */
#pragma omp parallel
  {
    REAL* a = (REAL*)malloc(sizeof(REAL) * (size_t)(4 * Fm + 2 * d + 2 * E));
    REAL *u = a + Fm, *h = u + Fm, *dh = h + Fm, *o = dh + Fm, *dov = o + d, *dp = dov + d;
#pragma omp for schedule(dynamic, 8)
    for (int t = 0; t < T; ++t) {
      const REAL* xt = x + (size_t)t * d;
      const REAL* dyt = dy + (size_t)t * d;
      const REAL* p = probs + (size_t)t * E;
      const int32_t* idx = topk_idx + (size_t)t * k;
      const REAL* g = gate + (size_t)t * k;
      REAL* dxt = dx + (size_t)t * d;
      REAL* dz = dlogits + (size_t)t * E;
      for (int i = 0; i < d; ++i) dxt[i] = 0;
      for (int e = 0; e < E; ++e) dp[e] = 0;
      for (int j = 0; j < k; ++j) {
        REAL* dg = dgate + (size_t)t * k + j;
        *dg = 0;
        int s = slot_of[idx[j]];
        if (s < 0) continue; /* ghost path does not exist in the graph */
        const REAL *wg = w_gate ? w_gate + (size_t)s * F * d : NULL, *wu = w_up + (size_t)s * F * d, *wd = w_down + (size_t)s * d * F;
        expert_fwd_(expert_fn, xt, d, F, wg, wu, wd, a, u, h, o);
        *dg = dot_(dyt, o, d);                      /* y += g o  =>  dg = <dy, o> */
        for (int i = 0; i < d; ++i) dov[i] = g[j] * dyt[i]; /*            do = g dy */
        expert_bwd_(expert_fn, xt, dov, d, F, wg, wu, wd, a, u, h, dh, dxt, NULL, NULL, NULL);
      }
      for (int s = 0; s < n_sh; ++s)
        expert_bwd_(expert_fn, xt, dyt, d, F_sh, sh_gate ? sh_gate + (size_t)s * F_sh * d : NULL, sh_up + (size_t)s * F_sh * d,
                    sh_down + (size_t)s * d * F_sh, a, u, h, dh, dxt, NULL, NULL, NULL);
      /* gate rule backward: dp from dg */
      if (gate_rule == RULE_DROP_ONLY) {
        for (int j = 0; j < k; ++j)
          if (slot_of[idx[j]] >= 0) dp[idx[j]] = dgate[(size_t)t * k + j];
      } else {
        /* g_j = p_j / s, s over the normalising set N (all k selected | kept only):
         * dp_j' = [j' kept] dg_j'/s - (sum_{j kept} dg_j g_j)/s   for j' in N */
        REAL ssum = 0, dgg = 0;
        for (int j = 0; j < k; ++j) {
          int kept = slot_of[idx[j]] >= 0;
          if (gate_rule == RULE_RENORM_TOPK || kept) ssum += p[idx[j]];
          if (kept) dgg += dgate[(size_t)t * k + j] * g[j];
        }
        for (int j = 0; j < k; ++j) {
          int kept = slot_of[idx[j]] >= 0;
          if (!(gate_rule == RULE_RENORM_TOPK || kept)) continue;
          if (ssum > 0) dp[idx[j]] = ((kept ? dgate[(size_t)t * k + j] : (REAL)0) - dgg) / ssum;
        }
      }
      /* gate function backward, then /tau (bias gets no gradient: it is a test device, R8) */
      if (gate_fn == GATE_SIGMOID) {
        for (int e = 0; e < E; ++e) dz[e] = dp[e] * p[e] * ((REAL)1 - p[e]) / (REAL)tau;
      } else {
        REAL pd = 0;
        for (int e = 0; e < E; ++e) pd += p[e] * dp[e];
        for (int e = 0; e < E; ++e) dz[e] = p[e] * (dp[e] - pd) / (REAL)tau;
      }
      /* z = x W_r / tau: dx += W_r dz (dz already carries 1/tau) */
      for (int i = 0; i < d; ++i) {
        REAL s = 0;
        for (int e = 0; e < E; ++e) s += w_r[(size_t)i * E + e] * dz[e];
        dxt[i] += s;
      }
    }
    free(a);
  }

  /* dW_r = x^T dz */
#pragma omp parallel for schedule(static)
  for (int i = 0; i < d; ++i) {
    REAL* row = dw_router + (size_t)i * E;
    for (int e = 0; e < E; ++e) row[e] = 0;
    for (int t = 0; t < T; ++t) axpy_(x[(size_t)t * d + i], dlogits + (size_t)t * E, row, E);
  }

  /* Phase 2, per resident slot: weight gradients over that slot's rows in row order.
   * "each worker responsible solely for updating its local experts". */
#pragma omp parallel
  {
    REAL* a = (REAL*)malloc(sizeof(REAL) * (size_t)(4 * Fm + d));
    REAL *u = a + Fm, *h = u + Fm, *dh = h + Fm, *dov = dh + Fm;
#pragma omp for schedule(dynamic, 1)
    for (int s = 0; s < n_res; ++s) {
      const REAL *wg = w_gate ? w_gate + (size_t)s * F * d : NULL, *wu = w_up + (size_t)s * F * d, *wd = w_down + (size_t)s * d * F;
      REAL *dwg = dw_gate ? dw_gate + (size_t)s * F * d : NULL, *dwu = dw_up + (size_t)s * F * d, *dwd = dw_down + (size_t)s * d * F;
      if (dwg) memset(dwg, 0, sizeof(REAL) * (size_t)F * d);
      memset(dwu, 0, sizeof(REAL) * (size_t)F * d);
      memset(dwd, 0, sizeof(REAL) * (size_t)F * d);
      for (int r = offsets[s]; r < offsets[s + 1]; ++r) {
        int t = row_token[r], j = -1;
        for (int jj = 0; jj < k; ++jj)
          if (topk_idx[(size_t)t * k + jj] == resident_ids[s]) j = jj;
        REAL gj = gate[(size_t)t * k + j];
        for (int i = 0; i < d; ++i) dov[i] = gj * dy[(size_t)t * d + i];
        expert_bwd_(expert_fn, x + (size_t)t * d, dov, d, F, wg, wu, wd, a, u, h, dh, NULL, dwg, dwu, dwd);
      }
    }
    free(a);
  }
  /* shared experts: every token, gate 1 */
  for (int s = 0; s < n_sh; ++s) {
    const REAL *wg = sh_gate ? sh_gate + (size_t)s * F_sh * d : NULL, *wu = sh_up + (size_t)s * F_sh * d, *wd = sh_down + (size_t)s * d * F_sh;
    REAL *dwg = d_sh_gate ? d_sh_gate + (size_t)s * F_sh * d : NULL, *dwu = d_sh_up + (size_t)s * F_sh * d, *dwd = d_sh_down + (size_t)s * d * F_sh;
    size_t n = (size_t)F_sh * d;
    if (dwg) memset(dwg, 0, sizeof(REAL) * n);
    memset(dwu, 0, sizeof(REAL) * n);
    memset(dwd, 0, sizeof(REAL) * n);
#pragma omp parallel
    {
      REAL* a = (REAL*)malloc(sizeof(REAL) * (size_t)(4 * Fm));
      REAL *u = a + Fm, *h = u + Fm, *dh = h + Fm;
      REAL* loc = (REAL*)calloc(3 * n, sizeof(REAL));
#pragma omp for schedule(static)
      for (int t = 0; t < T; ++t)
        expert_bwd_(expert_fn, x + (size_t)t * d, dy + (size_t)t * d, d, F_sh, wg, wu, wd, a, u, h, dh, NULL, loc, loc + n, loc + 2 * n);
#pragma omp critical
      {
        if (dwg) axpy_((REAL)1, loc, dwg, (int)n);
        axpy_((REAL)1, loc + n, dwu, (int)n);
        axpy_((REAL)1, loc + 2 * n, dwd, (int)n);
      }
      free(loc);
      free(a);
    }
  }
  free(slot_of);
  return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Sampled weight gradients for the full-size parity tests (outputs "the oracle can compute one by one"):
 * for resident slot s and each sampled hidden index f = f_idx[q], over ALL rows of the slot,
 *   dW_gate[s,f,:] = sum_r da_rf x_r,  dW_up[s,f,:] = sum_r du_rf x_r,  dW_down[s,:,f] = sum_r do_r h_rf
 * with do_r = g_r dy_t(r), dh_rf = <do_r, W_down[:,f]>, a_rf = <W_gate[f,:], x_r>, u_rf = <W_up[f,:], x_r>,
 * h_rf = silu(a_rf) u_rf, da = dh u s (1 + a (1 - s)), du = dh a s   (same formulas as expert_bwd_, one f at a time).
 * Outputs [n_f, d] each.  Pinned against oracle_moe_bwd in tests/test_oracle_pins.py.
 * ---------------------------------------------------------------------------------------------- */
int oracle_dw_sample(int d, int k, int F, int expert_fn, const REAL* x, const REAL* dy, const int32_t* topk_idx, const REAL* gate,
                     int resident_id, int row_begin, int row_end, const int32_t* row_token,
                     const REAL* wg, const REAL* wu, const REAL* wd, /* this slot's [F,d], [F,d], [d,F] */
                     const int32_t* f_idx, int n_f, REAL* dwg_rows, REAL* dwu_rows, REAL* dwd_cols) {
#pragma omp parallel for schedule(static)
  for (int q = 0; q < n_f; ++q) {
    const int f = f_idx[q];
    REAL *og = dwg_rows + (size_t)q * d, *ou = dwu_rows + (size_t)q * d, *od = dwd_cols + (size_t)q * d;
    for (int i = 0; i < d; ++i) og[i] = ou[i] = od[i] = 0;
    for (int r = row_begin; r < row_end; ++r) {
      const int t = row_token[r];
      int j = -1;
      for (int jj = 0; jj < k; ++jj)
        if (topk_idx[(size_t)t * k + jj] == resident_id) j = jj;
      const REAL g = gate[(size_t)t * k + j];
      const REAL *xt = x + (size_t)t * d, *dyt = dy + (size_t)t * d;
      const int silu = expert_fn == EXPERT_SILU; /* SiLU form: a = W_up x, u = 1, the gradient of W_up is da x */
      REAL a = silu ? dot_(wu + (size_t)f * d, xt, d) : dot_(wg + (size_t)f * d, xt, d);
      REAL u = silu ? (REAL)1 : dot_(wu + (size_t)f * d, xt, d);
      REAL sg = sigmoid_(a), h = a * sg * u, dh = 0;
      for (int i = 0; i < d; ++i) dh += g * dyt[i] * wd[(size_t)i * F + f];
      REAL da = dh * u * sg * ((REAL)1 + a * ((REAL)1 - sg)), du = dh * a * sg;
      if (silu) {
        axpy_(da, xt, ou, d);
      } else {
        axpy_(da, xt, og, d);
        axpy_(du, xt, ou, d);
      }
      axpy_(g * h, dyt, od, d);
    }
  }
  return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Step 10: resident-delta pack, always fp32 (BASELINE.json config 4 "fp32 resident-delta pack").
 * payload block b (b-th entry of pack_slots, or slot b if pack_slots == NULL) =
 *   [ w_start_gate - w_now_gate | w_start_up - w_now_up | w_start_down - w_now_down ]  of that slot
 * (PAPER.md:253 payload = the expert's projections; 824 Alg. 2 l.19; sign = round start minus local,
 * DESIGN.md R10).
 * ---------------------------------------------------------------------------------------------- */
int oracle_pack_resident_deltas(const float* now_gate, const float* now_up, const float* now_down,
                                const float* start_gate, const float* start_up, const float* start_down,
                                int n_res, int64_t elems_gate, int64_t elems_up, int64_t elems_down,
                                const int32_t* pack_slots, int n_pack, float* payload) {
  int64_t block = elems_gate + elems_up + elems_down;
  for (int b = 0; b < n_pack; ++b) {
    int s = pack_slots ? pack_slots[b] : b;
    if (s < 0 || s >= n_res) return -1;
    float* out = payload + (size_t)b * block;
    for (int64_t i = 0; i < elems_gate; ++i) out[i] = start_gate[(size_t)s * elems_gate + i] - now_gate[(size_t)s * elems_gate + i];
    out += elems_gate;
    for (int64_t i = 0; i < elems_up; ++i) out[i] = start_up[(size_t)s * elems_up + i] - now_up[(size_t)s * elems_up + i];
    out += elems_up;
    for (int64_t i = 0; i < elems_down; ++i) out[i] = start_down[(size_t)s * elems_down + i] - now_down[(size_t)s * elems_down + i];
  }
  return 0;
}
