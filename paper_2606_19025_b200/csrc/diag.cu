// Diagnostics around the routing step: validation of the resident set (the one entry point that synchronises) and the
// routing statistics the paper names as standard diagnostics ("routing entropy, load coefficients of variation,
// and overflow rates"; "the actual frequency of the token assignments to ghost experts against the total number
// of assignments").
#include <math.h>
#include <stdio.h>

#include <vector>

#include "common.cuh"

namespace fomoe {

// load[e] = number of (token, j) assignments to expert e over ALL E experts (ghosts included); load[E] = tokens with no kept
// pair; load[E + 1] = block ticket.  The last block to finish turns the histogram into the statistics (fixed order: e ascending).
__global__ void __launch_bounds__(256)
routing_stats_kernel(const int32_t* __restrict__ topk_idx, const int32_t* __restrict__ pair_row, int T, int k, int E,
                     int32_t* __restrict__ load, float* __restrict__ stats) {
  extern __shared__ int32_t sh[];   // [E + 1]
  for (int i = threadIdx.x; i <= E; i += blockDim.x) sh[i] = 0;
  __syncthreads();
  for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < T; t += gridDim.x * blockDim.x) {
    bool any = false;
    for (int j = 0; j < k; ++j) {
      const int e = topk_idx[(size_t)t * k + j];
      if (e >= 0 && e < E) atomicAdd(&sh[e], 1);
      any |= pair_row[(size_t)t * k + j] >= 0;
    }
    if (!any) atomicAdd(&sh[E], 1);
  }
  __syncthreads();
  for (int i = threadIdx.x; i <= E; i += blockDim.x)
    if (sh[i]) atomicAdd(&load[i], sh[i]);
  __threadfence();
  __shared__ bool last;
  __syncthreads();
  if (threadIdx.x == 0) last = atomicAdd(&load[E + 1], 1) == (int)gridDim.x - 1;
  __syncthreads();
  if (!last || threadIdx.x != 0) return;
  __threadfence();
  const volatile int32_t* ld = load;
  const double total = (double)T * k;
  double mean = total / E, var = 0.0, ent = 0.0;
  int mx = 0, mn = 0x7fffffff;
  for (int e = 0; e < E; ++e) {
    const int c = ld[e];
    const double dlt = c - mean;
    var += dlt * dlt;
    if (c > 0) { const double f = c / total; ent -= f * log(f); }
    mx = max(mx, c);
    mn = min(mn, c);
  }
  var /= E;
  stats[FOMOE_STAT_LOAD_CV] = total > 0 ? (float)(sqrt(var) / mean) : 0.f;
  stats[FOMOE_STAT_ROUTING_ENTROPY] = (float)ent;
  stats[FOMOE_STAT_ZERO_KEPT_TOKENS] = T > 0 ? (float)ld[E] / (float)T : 0.f;
  stats[FOMOE_STAT_MAX_LOAD] = (float)mx;
  stats[FOMOE_STAT_MIN_LOAD] = E > 0 ? (float)mn : 0.f;
}

// kept / ghost fractions need the resident slots: counts[n_res] sums to P
__global__ void routing_stats_kept_kernel(const int32_t* __restrict__ offsets, int n_res, int T, int k, float* __restrict__ stats) {
  const double total = (double)T * k;
  const double kept = total > 0 ? offsets[n_res] / total : 0.0;
  stats[FOMOE_STAT_KEPT_FRACTION] = (float)kept;
  stats[FOMOE_STAT_GHOST_FRACTION] = total > 0 ? (float)(1.0 - kept) : 0.f;
}

int launch_routing_stats(const fomoe_config& c, const fomoe_route_state& r, int n_res, int32_t* load, float* stats, cudaStream_t st) {
  FOMOE_CUDA_OK(cudaMemsetAsync(load, 0, sizeof(int32_t) * (size_t)(c.E + 2), st));
  FOMOE_CUDA_OK(cudaMemsetAsync(stats, 0, sizeof(float) * FOMOE_N_STATS, st));
  int grid = ceil_div(c.T > 0 ? c.T : 1, 256);
  if (grid > num_sms() * 4) grid = num_sms() * 4;
  routing_stats_kernel<<<grid, 256, sizeof(int32_t) * (size_t)(c.E + 1), st>>>(r.topk_idx, r.pair_row, c.T, c.top_k, c.E, load, stats);
  FOMOE_LAUNCH_OK("routing_stats_kernel");
  routing_stats_kept_kernel<<<1, 1, 0, st>>>(r.offsets, n_res, c.T, c.top_k, stats);
  FOMOE_LAUNCH_OK("routing_stats_kept_kernel");
  return FOMOE_OK;
}

// Synchronising check of the CONTENT of resident_ids (fomoe_route cannot afford it): range, strictly ascending (hence unique).
int validate_resident(const int32_t* resident_ids, int n_res, int E, cudaStream_t st, char* msg, size_t msg_len) {
  if (n_res == 0) return FOMOE_OK;
  std::vector<int32_t> h((size_t)n_res);
  FOMOE_CUDA_OK(cudaMemcpyAsync(h.data(), resident_ids, sizeof(int32_t) * (size_t)n_res, cudaMemcpyDeviceToHost, st));
  FOMOE_CUDA_OK(cudaStreamSynchronize(st));
  for (int i = 0; i < n_res; ++i) {
    if (h[i] < 0 || h[i] >= E) {
      snprintf(msg, msg_len, "resident_ids[%d] = %d is outside [0, %d)", i, h[i], E);
      return FOMOE_ERR_BADARG;
    }
    if (i > 0 && h[i] <= h[i - 1]) {
      snprintf(msg, msg_len, "resident_ids[%d] = %d after %d: ids must be strictly ascending (%s)", i, h[i], h[i - 1],
               h[i] == h[i - 1] ? "duplicate" : "unsorted");
      return FOMOE_ERR_BADARG;
    }
  }
  return FOMOE_OK;
}

}  // namespace fomoe
