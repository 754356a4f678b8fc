// Tensor-core router for bf16 tokens (rows F1-F4 of SURVEY.md §8(a), plus the per-block histogram of row F5).
//
// logits = x W_r is a [T,d] x [d,E] contraction with fp32 W_r and a bit-exactness bar on the top-k decision (margins of
// 1e-4), so W_r is split into 3 (or, for E > 80, 2) bf16 pieces  W = hi + mid + lo  (each piece the bf16 rounding of the
// running residual): x is bf16-exact, every product x*piece is exact in fp32, the pieces ride in one tcgen05.mma as
// extra N columns [hi | mid | lo] and are added in fp32 in the epilogue.  That keeps the router on the HBM roofline
// (x is read once by TMA) instead of being fp32-ALU bound at E >= 64.
//
// Epilogue: one thread per token row reads its logits straight from tensor memory (three light passes: max + top-k
// insertion, softmax denominator, probabilities), applies the residency mask and the gate rule,
// and adds its kept pairs to the block's per-slot histogram.  One CTA per 128-token tile.
#include "common.cuh"
#include "umma_ptx.cuh"

namespace fomoe {
namespace {

constexpr int kRStages = 4;
constexpr int kRThreads = 256;

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
  uint32_t* r = reinterpret_cast<uint32_t*>(v);
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                 "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr));
}

struct RouteUmmaParams {
  int T, d, E, Epad, pieces, NP, k, gate_fn, gate_rule, n_res;
  float inv_tau;
  const float* bias;
  const int32_t* slot_of;
  float* probs;
  int32_t* topk_idx;
  float* gate;
  int32_t* blk_hist;  // [gridDim.x, n_res]
};

// slot_of[e] and the bf16 split of W_r: wr_split[i, piece*Epad + e], zero elsewhere (row stride NP); also presets
// row_token / prow_token to -1 (rows that no kept pair claims).
__global__ void route_prep_kernel(const int32_t* __restrict__ resident_ids, int n_res, int E, int32_t* __restrict__ slot_of,
                                  const float* __restrict__ w_r, int d, int Epad, int pieces, int NP, bf16* __restrict__ wr_split,
                                  int32_t* __restrict__ row_token, long n_row_token, int32_t* __restrict__ prow_token, long n_prow_token) {
  pdl_launch_dependents();
  pdl_wait();
  const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  for (long i = idx; i < n_row_token; i += (long)gridDim.x * blockDim.x) row_token[i] = -1;
  for (long i = idx; i < n_prow_token; i += (long)gridDim.x * blockDim.x) prow_token[i] = -1;
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

template <int KMAX>
__global__ void __launch_bounds__(kRThreads, 1)
route_umma_kernel(const __grid_constant__ CUtensorMap map_x, const __grid_constant__ CUtensorMap map_w, const RouteUmmaParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const int b_bytes = p.NP * 128, stage_bytes = 16384 + b_bytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kRStages * stage_bytes);
  uint64_t* full_bar = bars;
  uint64_t* empty_bar = bars + kRStages;
  uint64_t* tfull_bar = bars + 2 * kRStages;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * kRStages + 1);
  int32_t* s_slot = reinterpret_cast<int32_t*>(bars + 2 * kRStages + 2);  // [E]
  int32_t* s_hist = s_slot + kMaxE;                                       // [n_res]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m0 = blockIdx.x * 128;
  const int num_kb = p.d / 64;
  const uint32_t tmem_cols = p.NP <= 64 ? 64u : p.NP <= 128 ? 128u : 256u;

  pdl_launch_dependents();
  for (int i = threadIdx.x; i < p.n_res; i += kRThreads) s_hist[i] = 0;
  if (warp == 0 && lane == 0) { prefetch_tmap(&map_x); prefetch_tmap(&map_w); }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < kRStages; ++i) { mbar_init(smem_u32(&full_bar[i]), 1); mbar_init(smem_u32(&empty_bar[i]), 1); }
    mbar_init(smem_u32(tfull_bar), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(tmem_cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  pdl_wait();   // everything above touches only shared / tensor memory
  for (int i = threadIdx.x; i < p.E; i += kRThreads) s_slot[i] = p.slot_of[i];
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int kb = 0; kb < num_kb; ++kb) {
        mbar_wait(smem_u32(&empty_bar[stage]), phase ^ 1);
        const uint32_t sa = smem_u32(smem + stage * stage_bytes), sb = sa + 16384, fb = smem_u32(&full_bar[stage]);
        mbar_expect_tx(fb, stage_bytes);
        tma_load_2d(sa, &map_x, fb, kb * 64, m0);
        for (int j = 0; j < p.NP / 64; ++j) tma_load_2d(sb + j * 8192, &map_w, fb, 64 * j, kb * 64);
        if (++stage == kRStages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 1) {
    // D fp32, A/B bf16, A K-major, B MN-major, M = 128, N = NP
    const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | (1u << 16) | ((uint32_t)(p.NP >> 3) << 17) | ((128u >> 4) << 24);
    int stage = 0;
    uint32_t phase = 0;
    for (int kb = 0; kb < num_kb; ++kb) {
      mbar_wait(smem_u32(&full_bar[stage]), phase);
      tc_fence_after();
      if (lane == 0) {
        const uint32_t sa = smem_u32(smem + stage * stage_bytes), sb = sa + 16384;
#pragma unroll
        for (int k = 0; k < 4; ++k)
          umma_bf16(tmem_base, make_desc(sa + k * 32, 16, 1024), make_desc(sb + k * 2048, 8192, 1024), idesc, (kb | k) != 0 ? 1u : 0u);
        umma_commit(smem_u32(&empty_bar[stage]));
        if (kb == num_kb - 1) umma_commit(smem_u32(tfull_bar));
      }
      __syncwarp();
      if (++stage == kRStages) { stage = 0; phase ^= 1; }
    }
  } else if (warp >= 4) {
    const int q = warp & 3;
    const int t = m0 + q * 32 + lane;
    const bool row_ok = t < p.T;
    const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16);
    const int E = p.E, Epad = p.Epad;
    const bool three = p.pieces == 3;
    mbar_wait(smem_u32(tfull_bar), 0);
    tc_fence_after();

    // logits of 16 experts starting at c0 (identical arithmetic in every pass)
    auto load_z = [&](int c0, float (&z)[16]) {
      float md[16], lo[16];
      tmem_ld16(taddr + c0, z);
      tmem_ld16(taddr + Epad + c0, md);
      if (three) tmem_ld16(taddr + 2 * Epad + c0, lo);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        float s = z[i] + md[i];
        if (three) s += lo[i];
        z[i] = s * p.inv_tau + (p.bias && c0 + i < E ? p.bias[c0 + i] : 0.f);
      }
    };

    // pass 1: running max and top-KMAX list (descending, ties -> lower id: ascending scan + strict '>')
    float tv[KMAX];
    int ti[KMAX];
#pragma unroll
    for (int j = 0; j < KMAX; ++j) { tv[j] = -INFINITY; ti[j] = kMaxE; }
    float mx = -INFINITY;
    for (int c0 = 0; c0 < Epad; c0 += 16) {
      float z[16];
      load_z(c0, z);
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        if (c0 + i < E) {
          float cv = z[i];
          int ci = c0 + i;
          mx = fmaxf(mx, cv);
          if (cv > tv[KMAX - 1]) {
            bool ins = false;
#pragma unroll
            for (int j = 0; j < KMAX; ++j) {
              const bool gt = ins || cv > tv[j];
              const float ov = tv[j];
              const int oi = ti[j];
              tv[j] = gt ? cv : ov;
              ti[j] = gt ? ci : oi;
              cv = gt ? ov : cv;
              ci = gt ? oi : ci;
              ins = gt;
            }
          }
        }
      }
    }
    // pass 2 (softmax): denominator
    float inv_s = 1.f;
    if (p.gate_fn == FOMOE_GATE_SOFTMAX) {
      float s = 0.f;
      for (int c0 = 0; c0 < Epad; c0 += 16) {
        float z[16];
        load_z(c0, z);
#pragma unroll
        for (int i = 0; i < 16; ++i)
          if (c0 + i < E) s += expf(z[i] - mx);
      }
      inv_s = 1.0f / s;
    }
    auto prob_of = [&](float z) { return p.gate_fn == FOMOE_GATE_SOFTMAX ? expf(z - mx) * inv_s : 1.0f / (1.0f + expf(-z)); };
    // pass 3: probabilities
    for (int c0 = 0; c0 < Epad; c0 += 16) {
      float z[16];
      load_z(c0, z);
#pragma unroll
      for (int i = 0; i < 16; ++i) z[i] = prob_of(z[i]);
      if (row_ok) {
        float* dst = p.probs + (size_t)t * E + c0;
        if ((E & 3) == 0) {
#pragma unroll
          for (int v = 0; v < 4; ++v)
            if (c0 + 4 * v < E) *reinterpret_cast<float4*>(dst + 4 * v) = make_float4(z[4 * v], z[4 * v + 1], z[4 * v + 2], z[4 * v + 3]);
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i)
            if (c0 + i < E) dst[i] = z[i];
        }
      }
    }
    // residency mask, gate rule, outputs, per-slot histogram
    if (row_ok) {
      float pj[KMAX];
      int sl[KMAX];
      float s_all = 0.f, s_kept = 0.f;
#pragma unroll
      for (int j = 0; j < KMAX; ++j) {
        pj[j] = 0.f;
        sl[j] = -1;
        if (j < p.k) {
          pj[j] = prob_of(tv[j]);
          sl[j] = s_slot[ti[j]];
          s_all += pj[j];
          if (sl[j] >= 0) s_kept += pj[j];
        }
      }
#pragma unroll
      for (int j = 0; j < KMAX; ++j) {
        if (j < p.k) {
          float g = 0.f;
          if (sl[j] >= 0) {
            g = p.gate_rule == FOMOE_DROP_ONLY ? pj[j] : p.gate_rule == FOMOE_RENORM_TOPK ? pj[j] / s_all : pj[j] / s_kept;
            atomicAdd(&s_hist[sl[j]], 1);
          }
          p.topk_idx[(size_t)t * p.k + j] = ti[j];
          p.gate[(size_t)t * p.k + j] = g;
        }
      }
    }
    tc_fence_before();
    asm volatile("bar.sync 1, 128;" ::: "memory");  // the four epilogue warps
    for (int i = threadIdx.x - 128; i < p.n_res; i += 128) p.blk_hist[(size_t)blockIdx.x * p.n_res + i] = s_hist[i];
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(tmem_cols) : "memory");
}

}  // namespace

bool route_umma_supported(const fomoe_config& c) {
  return c.dtype == FOMOE_BF16 && c.d_model % 64 == 0 && c.E <= 128 && c.top_k <= 8 && c.T > 0;
}

// x [T,d] bf16.  Writes slot_of, probs, topk_idx, gate and blk_hist (one row per 128-token block).
int launch_route_umma(const fomoe_config& c, const void* x, const float* w_router, const float* bias, const int32_t* resident_ids,
                      int n_res, const fomoe_route_state& out, const RouteWs& ws, cudaStream_t st) {
  const int E = c.E, d = c.d_model;
  const int Epad = (E + 15) / 16 * 16;
  const int pieces = 3 * Epad <= 256 ? 3 : 2;
  const int NP = (pieces * Epad + 63) / 64 * 64;
  {
    const long n = (long)d * NP > E ? (long)d * NP : E;
    FOMOE_CUDA_OK(launch_pdl(route_prep_kernel, (unsigned)((n + 255) / 256), 256, 0, st, resident_ids, n_res, E, ws.slot_of, w_router, d,
                             Epad, pieces, NP, (bf16*)ws.wr_split, out.row_token, (long)c.T * c.top_k, ws.prow_token, (long)ws.R_cap));
    FOMOE_LAUNCH_OK("route_prep_kernel");
  }
  CUtensorMap mx, mw;
  MAP_OK(make_map(&mx, x, d, c.T, d, 128));
  MAP_OK(make_map(&mw, ws.wr_split, NP, d, NP, 64));
  RouteUmmaParams p{c.T, d, E, Epad, pieces, NP, c.top_k, c.gate_fn, c.gate_rule, n_res, 1.0f / c.temperature, bias, ws.slot_of,
                    out.probs, out.topk_idx, out.gate, ws.blk_hist};
  const int smem = kRStages * (16384 + NP * 128) + 1024 + 8 * (2 * kRStages + 2) + 4 * (kMaxE + kMaxE);
  const int grid = ceil_div(c.T, 128);
#define ROUTE_UMMA_CASE(KM)                                                                                        \
  {                                                                                                                \
    FOMOE_CUDA_OK(cudaFuncSetAttribute(route_umma_kernel<KM>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)); \
    FOMOE_CUDA_OK(launch_pdl(route_umma_kernel<KM>, grid, kRThreads, smem, st, mx, mw, p));                        \
  }
  if (c.top_k <= 2) ROUTE_UMMA_CASE(2)
  else if (c.top_k <= 4) ROUTE_UMMA_CASE(4)
  else ROUTE_UMMA_CASE(8)
#undef ROUTE_UMMA_CASE
  FOMOE_LAUNCH_OK("route_umma_kernel");
  return FOMOE_OK;
}

}  // namespace fomoe
