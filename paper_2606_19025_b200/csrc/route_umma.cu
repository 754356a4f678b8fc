// Tensor-core router for bf16 tokens (rows F1-F4 of SURVEY.md §8(a), plus the per-block histogram of row F5).
//
// logits = x W_r is a [T,d] x [d,E] contraction with fp32 W_r and a bit-exactness bar on the top-k decision (margins of
// 1e-4), so W_r is split into 3 (or, for E > 80, 2) bf16 pieces  W = hi + mid + lo  (each piece the bf16 rounding of the
// running residual): x is bf16-exact, every product x*piece is exact in fp32, the pieces ride in one tcgen05.mma as
// extra N columns [hi | mid | lo] and are added in fp32 in the epilogue.  That keeps the router on the HBM roofline
// (x is read once by TMA) instead of being fp32-ALU bound at E >= 64.
//
// This file holds the preparation kernel (slot map, the split of W_r, bf16 W_r for the backward, row-map presets); the
// contraction and its epilogue (gate, top-k, residency mask, gate rule, per-block histogram: PAPER.md:157-159, 519, 593)
// are the ROUTE mode of the persistent CTA-pair kernel in umma_gemm.cu.
#include "common.cuh"
#include "umma_ptx.cuh"

namespace fomoe {
namespace {

// slot_of[e] and the bf16 split of W_r: wr_split[i, piece*Epad + e], zero elsewhere (row stride NP); also presets
// row_token / prow_token to -1 (rows that no kept pair claims).
__global__ void route_prep_kernel(const int32_t* __restrict__ resident_ids, int n_res, int E, int32_t* __restrict__ slot_of,
                                  const float* __restrict__ w_r, int d, int Epad, int pieces, int NP, bf16* __restrict__ wr_split,
                                  int32_t* __restrict__ row_token, long n_row_token, int32_t* __restrict__ prow_token, long n_prow_token,
                                  bf16* __restrict__ wr_bf, int Ez) {
  pdl_launch_dependents();
  pdl_wait();
  const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  for (long i = idx; i < n_row_token; i += (long)gridDim.x * blockDim.x) row_token[i] = -1;
  for (long i = idx; i < n_prow_token; i += (long)gridDim.x * blockDim.x) prow_token[i] = -1;
  for (long i = idx; i < (long)d * Ez; i += (long)gridDim.x * blockDim.x) {  // operand of the router backward (B7)
    const int r = (int)(i / Ez), e = (int)(i % Ez);
    wr_bf[i] = __float2bfloat16_rn(e < E ? w_r[(size_t)r * E + e] : 0.f);
  }
  if (idx < E) {
    int s = -1;
    for (int i = 0; i < n_res; ++i)
      if (resident_ids[i] == (int)idx) s = i;
    slot_of[idx] = s;
  }
  if (wr_split && idx < (long)d * NP) {
    const int i = (int)(idx / NP), col = (int)(idx % NP);
    const int piece = col / Epad, e = col % Epad;
    float out = 0.f;
    if (piece < pieces && e < E) {
      float r = w_r[(size_t)i * E + e];
      for (int pc = 0; pc < piece; ++pc) r -= __bfloat162float(__float2bfloat16_rn(r));  // exact in fp32
      out = r;
    }
    wr_split[idx] = __float2bfloat16_rn(out);
  }
}

}  // namespace

bool route_umma_supported(const fomoe_config& c) {
  return c.dtype == FOMOE_BF16 && c.d_model % 64 == 0 && c.E <= 128 && c.top_k <= kMaxK && c.T > 0;
}

// x [T,d] bf16.  Writes slot_of, probs, topk_idx, gate and blk_hist (one row per 128-token block).
int launch_route_umma(const fomoe_config& c, const void* x, const float* w_router, const float* bias, const int32_t* resident_ids,
                      int n_res, const fomoe_route_state& out, const RouteWs& ws, cudaStream_t st) {
  const int E = c.E, d = c.d_model;
  const int Epad = (E + 15) / 16 * 16;
  const int pieces = 3 * Epad <= 256 ? 3 : 2;
  const int NP = pieces * Epad <= 128 ? 128 : 256;   // accumulator columns of the CTA pair
  {
    const long n = (long)d * NP > E ? (long)d * NP : E;
    FOMOE_CUDA_OK(launch_pdl(route_prep_kernel, (unsigned)((n + 255) / 256), 256, 0, st, resident_ids, n_res, E, ws.slot_of, w_router, d,
                             Epad, pieces, NP, (bf16*)ws.wr_split, out.row_token, (long)c.T * c.top_k, ws.prow_token, (long)ws.R_cap,
                             (bf16*)ws.wr_bf, (E + 63) / 64 * 64));
    FOMOE_LAUNCH_OK("route_prep_kernel");
  }
  return umma_route(c, x, ws.wr_split, NP, Epad, pieces, bias, n_res, out, ws, st);
}

}  // namespace fomoe
