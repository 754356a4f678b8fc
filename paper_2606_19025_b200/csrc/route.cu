// Router GEMM + gate + top-k + residency mask + gate rule (rows F1-F4), and the histogram / prefix-scan /
// stable-scatter permutation (row F5) of SURVEY.md §8(a).  PAPER.md:159 (router over all E), 517-519 (Eq. 13-14),
// 595 (Eq. 17), 157-159 (skip-token).
#include "common.cuh"

namespace fomoe {

// ---------------------------------------------------------------------------------------------------------
// slot_of[e] = resident slot or -1
// ---------------------------------------------------------------------------------------------------------
__global__ void slot_map_kernel(const int32_t* __restrict__ resident_ids, int n_res, int E, int32_t* __restrict__ slot_of) {
  int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= E) return;
  int s = -1;
  for (int i = 0; i < n_res; ++i)
    if (resident_ids[i] == e) s = i;
  slot_of[e] = s;
}

// ---------------------------------------------------------------------------------------------------------
// Router: a block owns kTok = 32 tokens.  Phase 1: logits tile [32, E] by fp32 FMA (warp w accumulates experts
// w, w+8, ... for the 32 tokens: x from shared memory conflict-free, W_r broadcast).  Phase 2: one warp per token:
// gate function, k rounds of warp arg-max (ties -> lower expert id), residency mask, gate rule.
// ---------------------------------------------------------------------------------------------------------
constexpr int kTok = 32;
constexpr int kRouteThreads = 256;
constexpr int kRouteKC = 64;  // K chunk staged in shared memory

template <typename XT, int EPW>  // EPW = experts per warp = ceil(E / 8)
__global__ void __launch_bounds__(kRouteThreads)
route_kernel(const XT* __restrict__ x, const float* __restrict__ w_r, const float* __restrict__ bias,
             const int32_t* __restrict__ slot_of, int T, int d, int E, int k, int gate_fn, int gate_rule, float inv_tau, int forced_local,
             float* __restrict__ probs, int32_t* __restrict__ topk_idx, float* __restrict__ gate) {
  extern __shared__ float smem[];
  float* xs = smem;                            // [kTok][kRouteKC + 1]
  float* ws = xs + kTok * (kRouteKC + 1);      // [kRouteKC][E]
  float* zs = ws + kRouteKC * E;               // [kTok][E + 1]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int t0 = blockIdx.x * kTok;

  float acc[EPW];
#pragma unroll
  for (int i = 0; i < EPW; ++i) acc[i] = 0.f;

  for (int k0 = 0; k0 < d; k0 += kRouteKC) {
    const int kc = min(kRouteKC, d - k0);
    for (int i = tid; i < kTok * kRouteKC; i += kRouteThreads) {
      int tt = i / kRouteKC, kk = i % kRouteKC;
      float v = 0.f;
      if (t0 + tt < T && kk < kc) v = to_f32(x[(size_t)(t0 + tt) * d + k0 + kk]);
      xs[tt * (kRouteKC + 1) + kk] = v;
    }
    for (int i = tid; i < kRouteKC * E; i += kRouteThreads) {
      int kk = i / E, e = i % E;
      ws[i] = kk < kc ? w_r[(size_t)(k0 + kk) * E + e] : 0.f;
    }
    __syncthreads();
#pragma unroll 4
    for (int kk = 0; kk < kRouteKC; ++kk) {
      float xv = xs[lane * (kRouteKC + 1) + kk];
#pragma unroll
      for (int i = 0; i < EPW; ++i) {
        int e = warp + 8 * i;
        if (e < E) acc[i] = fmaf(xv, ws[kk * E + e], acc[i]);
      }
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < EPW; ++i) {
    int e = warp + 8 * i;
    // forced-local routing: the partitioned router has no column for a non-resident expert
    if (e < E) zs[lane * (E + 1) + e] = (forced_local && slot_of[e] < 0) ? -INFINITY : acc[i] * inv_tau + (bias ? bias[e] : 0.f);
  }
  __syncthreads();

  // phase 2: warp per token
  constexpr int kMaxPerLane = kMaxE / 32;
  for (int tt = warp; tt < kTok; tt += kRouteThreads / 32) {
    const int t = t0 + tt;
    if (t >= T) break;
    float z[kMaxPerLane], p[kMaxPerLane];
    float m = -INFINITY;
#pragma unroll
    for (int i = 0; i < kMaxPerLane; ++i) {
      int e = lane + 32 * i;
      z[i] = e < E ? zs[tt * (E + 1) + e] : -INFINITY;
      m = fmaxf(m, z[i]);
    }
    if (gate_fn == FOMOE_GATE_SIGMOID) {
#pragma unroll
      for (int i = 0; i < kMaxPerLane; ++i) p[i] = 1.0f / (1.0f + expf(-z[i]));
    } else {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
      float s = 0.f;
#pragma unroll
      for (int i = 0; i < kMaxPerLane; ++i) {
        p[i] = (lane + 32 * i) < E ? expf(z[i] - m) : 0.f;
        s += p[i];
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      float inv = 1.0f / s;
#pragma unroll
      for (int i = 0; i < kMaxPerLane; ++i) p[i] *= inv;
    }
#pragma unroll
    for (int i = 0; i < kMaxPerLane; ++i) {
      int e = lane + 32 * i;
      if (e < E) probs[(size_t)t * E + e] = p[i];
    }
    // k rounds of arg-max on z; a taken entry becomes -inf.  Tie -> lower expert id.
    float s_all = 0.f, s_kept = 0.f;
    float my_p = 0.f;   // lane j (< k) keeps p of the j-th selected expert
    int my_e = -1, my_slot = -1;
    for (int j = 0; j < k; ++j) {
      float bv = -INFINITY;
      int be = kMaxE;
#pragma unroll
      for (int i = 0; i < kMaxPerLane; ++i) {
        int e = lane + 32 * i;
        if (e < E && z[i] > bv) { bv = z[i]; be = e; }  // ascending e inside a lane: strict '>' keeps the lower id
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        float ov = __shfl_xor_sync(0xffffffffu, bv, o);
        int oe = __shfl_xor_sync(0xffffffffu, be, o);
        if (ov > bv || (ov == bv && oe < be)) { bv = ov; be = oe; }
      }
      // fewer than k logits compare greater than -inf (NaN / inf activations, a -inf bias): no candidate left.  Keep the id in
      // range so that nothing downstream indexes with the sentinel; such a pair carries the probability of that expert
      if (be >= E) be = E - 1;
      // owner lane marks it taken and publishes p
      float pe = 0.f;
#pragma unroll
      for (int i = 0; i < kMaxPerLane; ++i)
        if (lane + 32 * i == be) { pe = p[i]; z[i] = -INFINITY; }
      pe = __shfl_sync(0xffffffffu, pe, be & 31);
      int sl = slot_of[be];
      s_all += pe;
      if (sl >= 0) s_kept += pe;
      if (lane == j) { my_p = pe; my_e = be; my_slot = sl; }
    }
    if (lane < k) {
      float g = 0.f;
      if (my_slot >= 0)
        g = gate_rule == FOMOE_DROP_ONLY ? my_p : gate_rule == FOMOE_RENORM_TOPK ? my_p / s_all : my_p / s_kept;
      topk_idx[(size_t)t * k + lane] = my_e;
      gate[(size_t)t * k + lane] = g;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// Permutation.  Pairs are numbered p = t*k + j; a block owns the kPermTokens * k pairs of one 128-token router tile.
// ---------------------------------------------------------------------------------------------------------
__global__ void perm_hist_kernel(const int32_t* __restrict__ topk_idx, const int32_t* __restrict__ slot_of, long n_pairs,
                                 int pairs_per_blk, int n_res, int32_t* __restrict__ blk_hist) {
  extern __shared__ int32_t hist[];
  for (int i = threadIdx.x; i < n_res; i += blockDim.x) hist[i] = 0;
  __syncthreads();
  long p0 = (long)blockIdx.x * pairs_per_blk;
  for (int i = threadIdx.x; i < pairs_per_blk; i += blockDim.x) {
    long p = p0 + i;
    if (p < n_pairs) {
      int s = slot_of[topk_idx[p]];
      if (s >= 0) atomicAdd(&hist[s], 1);
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < n_res; i += blockDim.x) blk_hist[(size_t)blockIdx.x * n_res + i] = hist[i];
}

constexpr int kPermThreads = 256;

// Scan + scatter in ONE launch: every block re-derives, from the per-block histograms, its own exclusive base per slot and
// the slot totals (n_blk x n_res integers, L2-resident), the offsets by a warp scan over the slots, and then scatters its
// pairs; block 0 also publishes counts / offsets / padded offsets / K-range ends / tile maps.  Saves the single-block scan
// launch that sat on the critical path between the router and the gather.
__global__ void __launch_bounds__(kPermThreads)
perm_scan_scatter_kernel(const int32_t* __restrict__ topk_idx, const float* __restrict__ gate, const int32_t* __restrict__ slot_of,
                         const int32_t* __restrict__ blk_hist, int n_blk, long n_pairs, int pairs_per_blk, int k, int n_res,
                         int32_t* __restrict__ counts, int32_t* __restrict__ offsets, int32_t* __restrict__ pad_offsets,
                         int32_t* __restrict__ pad_end64, int32_t* __restrict__ n_mtiles, int32_t* __restrict__ tile_slot,
                         int32_t* __restrict__ pair_info, int32_t* __restrict__ row_token, int32_t* __restrict__ pair_row,
                         int32_t* __restrict__ prow_token, float* __restrict__ prow_gate, int32_t* __restrict__ prow_pair,
                         int32_t* __restrict__ pair_prow) {
  extern __shared__ int32_t sm[];
  __shared__ int32_t s_cnt[kMaxE], s_off[kMaxE + 1], s_pad[kMaxE + 1], s_pair[kMaxE + 1];
  pdl_launch_dependents();
  pdl_wait();
  int32_t* running = sm;                 // [n_res] rows of slot s taken by earlier blocks and by this block so far
  int32_t* warp_cnt = sm + n_res;        // [8][n_res]
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int n_warps = kPermThreads / 32;
  // (a) this block's exclusive base and the total of every slot.  The [n_blk, n_res] histogram is walked in memory order
  // (consecutive threads read consecutive words: every block reads all of it, so at T = 131072 the slot-per-warp walk with
  // its n_res-word stride took 198 us; this one 1/10 of that); integer adds, so the result does not depend on their order
  for (int i = threadIdx.x; i < n_res; i += kPermThreads) { running[i] = 0; s_cnt[i] = 0; }
  for (int i = threadIdx.x; i < 8 * n_res; i += kPermThreads) warp_cnt[i] = 0;
  __syncthreads();
  {
    const long n_hist = (long)n_blk * n_res, n_before = (long)blockIdx.x * n_res;
    if (kPermThreads % n_res == 0) {      // a thread meets one slot only: sums in registers, one shared-memory add at the end
      int base = 0, tot = 0;
      for (long i = threadIdx.x; i < n_hist; i += kPermThreads) {
        const int c = blk_hist[i];
        tot += c;
        if (i < n_before) base += c;
      }
      atomicAdd(&running[threadIdx.x % n_res], base);
      atomicAdd(&s_cnt[threadIdx.x % n_res], tot);
    } else {
      for (long i = threadIdx.x; i < n_hist; i += kPermThreads) {
        const int c = blk_hist[i];
        if (c == 0) continue;
        const int sidx = (int)(i % n_res);
        atomicAdd(&s_cnt[sidx], c);
        if (i < n_before) atomicAdd(&running[sidx], c);
      }
    }
  }
  __syncthreads();
  // (b) exclusive scans over the slots (warp 0): row offsets, tile-padded offsets, tile pairs
  if (warp == 0) {
    int off = 0, pad = 0, pairs = 0;
    for (int s0 = 0; s0 < n_res; s0 += 32) {
      const int s = s0 + lane;
      const int c = s < n_res ? s_cnt[s] : 0;
      const int tiles = (c + kTileM - 1) / kTileM;
      int ic = c, ip = tiles * kTileM, iq = (tiles + 1) / 2;
      const int pc = ip, qc = iq;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int vc = __shfl_up_sync(0xffffffffu, ic, o), vp = __shfl_up_sync(0xffffffffu, ip, o), vq = __shfl_up_sync(0xffffffffu, iq, o);
        if (lane >= o) { ic += vc; ip += vp; iq += vq; }
      }
      if (s < n_res) { s_off[s] = off + ic - c; s_pad[s] = pad + ip - pc; s_pair[s] = pairs + iq - qc; }
      off += __shfl_sync(0xffffffffu, ic, 31);
      pad += __shfl_sync(0xffffffffu, ip, 31);
      pairs += __shfl_sync(0xffffffffu, iq, 31);
    }
    if (lane == 0) { s_off[n_res] = off; s_pad[n_res] = pad; s_pair[n_res] = pairs; }
  }
  __syncthreads();
  if (blockIdx.x == 0) {   // publish
    for (int s = threadIdx.x; s < n_res; s += kPermThreads) {
      counts[s] = s_cnt[s];
      offsets[s] = s_off[s];
      pad_offsets[s] = s_pad[s];
      pad_end64[s] = s_pad[s] + (s_cnt[s] + 63) / 64 * 64;
    }
    if (threadIdx.x == 0) {
      offsets[n_res] = s_off[n_res];
      pad_offsets[n_res] = s_pad[n_res];
      n_mtiles[0] = s_pad[n_res] / kTileM;
      n_mtiles[1] = s_pad[n_res];
      n_mtiles[2] = s_pair[n_res];
    }
    for (int s = warp; s < n_res; s += n_warps) {
      const int t0 = s_pad[s] / kTileM, t1 = s_pad[s + 1] / kTileM;
      for (int i = t0 + lane; i < t1; i += 32) tile_slot[i] = s;
      for (int i = lane; i < s_pair[s + 1] - s_pair[s]; i += 32)
        pair_info[s_pair[s] + i] = 2 * (t0 + 2 * i) + (t0 + 2 * i + 1 < t1 ? 1 : 0);
    }
  }
  // (c) stable scatter of this block's pairs
  const long p0 = (long)blockIdx.x * pairs_per_blk;
  for (int it = 0; it < (pairs_per_blk + kPermThreads - 1) / kPermThreads; ++it) {
    const int ip = it * kPermThreads + threadIdx.x;
    const long p = ip < pairs_per_blk ? p0 + ip : n_pairs;   // out of this block's range -> inactive
    int s = -1;
    if (p < n_pairs) s = slot_of[topk_idx[p]];
    unsigned m = __match_any_sync(0xffffffffu, s);
    int rank_in_warp = __popc(m & ((1u << lane) - 1));
    if (s >= 0 && rank_in_warp == 0) warp_cnt[warp * n_res + s] = __popc(m);
    __syncthreads();
    if (p < n_pairs) {
      if (s >= 0) {
        int rank = running[s] + rank_in_warp;
        for (int w = 0; w < warp; ++w) rank += warp_cnt[w * n_res + s];
        int r = s_off[s] + rank, pr = s_pad[s] + rank;
        int t = (int)(p / k);
        row_token[r] = t;
        pair_row[p] = r;
        prow_token[pr] = t;
        prow_gate[pr] = gate[p];
        prow_pair[pr] = (int32_t)p;
        pair_prow[p] = pr;
      } else {
        pair_row[p] = -1;
        pair_prow[p] = -1;
      }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n_res; i += kPermThreads) {
      int add = 0;
      for (int w = 0; w < 8; ++w) { add += warp_cnt[w * n_res + i]; warp_cnt[w * n_res + i] = 0; }
      running[i] += add;
    }
    __syncthreads();
  }
}

template <typename XT>
static int launch_route_t(const fomoe_config& c, const XT* x, const float* w_router, const float* bias, const RouteWs& ws,
                          const fomoe_route_state& out, cudaStream_t st) {
  const int E = c.E;
  const int epw = ceil_div(E, 8);
  size_t smem = sizeof(float) * ((size_t)kTok * (kRouteKC + 1) + (size_t)kRouteKC * E + (size_t)kTok * (E + 1));
  dim3 grid(ceil_div(c.T, kTok));
  const float inv_tau = 1.0f / c.temperature;
#define ROUTE_CASE(N)                                                                                                   \
  {                                                                                                                     \
    auto kern = route_kernel<XT, N>;                                                                                    \
    FOMOE_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));                   \
    kern<<<grid, kRouteThreads, smem, st>>>(x, w_router, bias, ws.slot_of, c.T, c.d_model, E, c.top_k, c.gate_fn,        \
                                            c.gate_rule, inv_tau, c.route_mode == FOMOE_ROUTE_FORCED_LOCAL ? 1 : 0, out.probs, out.topk_idx, out.gate);                   \
  }
  if (epw <= 1) ROUTE_CASE(1)
  else if (epw <= 2) ROUTE_CASE(2)
  else if (epw <= 4) ROUTE_CASE(4)
  else if (epw <= 8) ROUTE_CASE(8)
  else if (epw <= 16) ROUTE_CASE(16)
  else if (epw <= 32) ROUTE_CASE(32)
  else ROUTE_CASE(64)
#undef ROUTE_CASE
  FOMOE_LAUNCH_OK("route_kernel");
  return FOMOE_OK;
}

int launch_route(const fomoe_config& c, const void* x, const float* w_router, const float* bias, const int32_t* resident_ids,
                 int n_res, const fomoe_route_state& out, const RouteWs& ws, cudaStream_t st) {
  const long n_pairs = (long)c.T * c.top_k;
  const int pairs_per_blk = kPermTokens * c.top_k;
  const int nr = n_res > 0 ? n_res : 1;
  const bool tc = c.T > 0 && !force_simt() && route_umma_supported(c);
  if (!tc) {  // (the tensor-core path fills these in its preparation kernel)
    FOMOE_CUDA_OK(cudaMemsetAsync(out.row_token, 0xFF, sizeof(int32_t) * (size_t)n_pairs, st));
    FOMOE_CUDA_OK(cudaMemsetAsync(ws.prow_token, 0xFF, sizeof(int32_t) * (size_t)ws.R_cap, st));
  }
  if (c.T == 0) {  // empty batch: all counts and offsets are zero, no tile in use
    if (n_res > 0) FOMOE_CUDA_OK(cudaMemsetAsync(out.counts, 0, sizeof(int32_t) * (size_t)n_res, st));
    FOMOE_CUDA_OK(cudaMemsetAsync(out.offsets, 0, sizeof(int32_t) * (size_t)(n_res + 1), st));
    FOMOE_CUDA_OK(cudaMemsetAsync(ws.pad_offsets, 0, sizeof(int32_t) * (size_t)(n_res + 1), st));
    FOMOE_CUDA_OK(cudaMemsetAsync(ws.n_mtiles, 0, sizeof(int32_t) * 4, st));
    FOMOE_CUDA_OK(cudaMemsetAsync(ws.pad_end64, 0, sizeof(int32_t) * (size_t)nr, st));
    return FOMOE_OK;
  }
  if (tc) {
    // tensor-core router: logits + gate + top-k + mask + per-block histogram in one kernel
    int rc = launch_route_umma(c, x, w_router, bias, resident_ids, n_res, out, ws, st);
    if (rc != FOMOE_OK) return rc;
  } else {
    slot_map_kernel<<<ceil_div(c.E, 128), 128, 0, st>>>(resident_ids, n_res, c.E, ws.slot_of);
    FOMOE_LAUNCH_OK("slot_map_kernel");
    int rc = c.dtype == FOMOE_BF16 ? launch_route_t<__nv_bfloat16>(c, (const __nv_bfloat16*)x, w_router, bias, ws, out, st)
                                   : launch_route_t<float>(c, (const float*)x, w_router, bias, ws, out, st);
    if (rc != FOMOE_OK) return rc;
    perm_hist_kernel<<<ws.n_blk, 256, sizeof(int32_t) * nr, st>>>(out.topk_idx, ws.slot_of, n_pairs, pairs_per_blk, n_res, ws.blk_hist);
    FOMOE_LAUNCH_OK("perm_hist_kernel");
  }
  FOMOE_CUDA_OK(launch_pdl(perm_scan_scatter_kernel, ws.n_blk, kPermThreads, sizeof(int32_t) * 9 * nr, st, out.topk_idx, out.gate, ws.slot_of,
                           ws.blk_hist, ws.n_blk, n_pairs, pairs_per_blk, c.top_k, n_res, out.counts, out.offsets, ws.pad_offsets, ws.pad_end64,
                           ws.n_mtiles, ws.tile_slot, ws.pair_info, out.row_token, out.pair_row, ws.prow_token, ws.prow_gate, ws.prow_pair,
                           ws.pair_prow));
  FOMOE_LAUNCH_OK("perm_scan_scatter_kernel");
  return FOMOE_OK;
}

}  // namespace fomoe
