// Row-wise, HBM-bound kernels around the expert GEMMs: gather of token rows into the tile-padded per-slot layout,
// gate-weighted combine (row F8, Eq. 13) and its backward (B1), gate backward (B6) and the final
// dx scatter-sum (B5).  All sums run in a fixed order (ascending j), so results are run-to-run identical.
#include "common.cuh"

namespace fomoe {

// 16-byte vector of V elements of T, held as fp32 in registers.
template <typename T, int V> struct Vec {
  float v[V];
  __device__ __forceinline__ void load(const T* p) {
    if constexpr (V == 1) {
      v[0] = to_f32(p[0]);
    } else if constexpr (sizeof(T) == 4) {
      float4 r = *reinterpret_cast<const float4*>(p);
      v[0] = r.x; v[1] = r.y; v[2] = r.z; v[3] = r.w;
    } else {
      uint4 r = *reinterpret_cast<const uint4*>(p);
      const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&r);
#pragma unroll
      for (int i = 0; i < 4; ++i) { float2 f = __bfloat1622float2(h[i]); v[2 * i] = f.x; v[2 * i + 1] = f.y; }
    }
  }
  __device__ __forceinline__ void store(T* p) const {
    if constexpr (V == 1) {
      p[0] = from_f32<T>(v[0]);
    } else if constexpr (sizeof(T) == 4) {
      *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
    } else {
      uint4 r;
      __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&r);
#pragma unroll
      for (int i = 0; i < 4; ++i) h[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]);
      *reinterpret_cast<uint4*>(p) = r;
    }
  }
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int i = 0; i < V; ++i) v[i] = 0.f;
  }
};

constexpr int kRowThreads = 128;
// CTAs of a row kernel: 16 per SM when the tensor is small (each CTA then loops over a few rows and the launch stays cheap),
// 64 per SM from ~24 M elements on (more rows in flight per SM: +5-10 % of HBM bandwidth on C3 / C5, measured)
static int row_grid(long rows, int d = 0) {
  const long cap = (rows * (long)d >= 24L * 1000 * 1000) ? (long)num_sms() * 64 : (long)num_sms() * 16;
  long g = rows < cap ? rows : cap;
  return (int)(g < 1 ? 1 : g);
}

// xp[r] = x[prow_token[r]] or 0 for a padding row; rows beyond the padded total are not touched.
template <typename T, int V>
__global__ void __launch_bounds__(kRowThreads)
gather_rows_kernel(const T* __restrict__ x, const int32_t* __restrict__ prow_token, const int32_t* __restrict__ n_mtiles, int d,
                   T* __restrict__ xp) {
  pdl_launch_dependents();
  pdl_wait();
  const int rows = n_mtiles[1];
  for (int r = blockIdx.x; r < rows; r += gridDim.x) {
    const int t = prow_token[r];
    for (int c = threadIdx.x * V; c < d; c += kRowThreads * V) {
      Vec<T, V> a;
      if (t >= 0) a.load(x + (size_t)t * d + c); else a.zero();
      a.store(xp + (size_t)r * d + c);
    }
  }
}

// y[t] = sum_{j, ascending} gate[t,j] * o[pair_prow[t,j]] (+ y_sh[t]); exactly 0 when nothing is kept.
template <typename T, int V>
__global__ void __launch_bounds__(kRowThreads)
combine_kernel(const T* __restrict__ o, const T* __restrict__ y_sh, const float* __restrict__ gate,
               const int32_t* __restrict__ pair_prow, int T_, int d, int k, int rpb, T* __restrict__ y) {
  pdl_launch_dependents();
  pdl_wait();
  // rpb token rows per CTA (narrow rows: d / V < kRowThreads would leave threads idle), kRowThreads / rpb threads each
  const int tpr = kRowThreads / rpb, sub = threadIdx.x / tpr, c0 = (threadIdx.x % tpr) * V;
  for (int t = blockIdx.x * rpb + sub; t < T_; t += gridDim.x * rpb) {
    for (int c = c0; c < d; c += tpr * V) {
      Vec<T, V> acc;
      if (y_sh) acc.load(y_sh + (size_t)t * d + c); else acc.zero();
      for (int j = 0; j < k; ++j) {
        const int r = pair_prow[(size_t)t * k + j];
        if (r < 0) continue;
        const float g = gate[(size_t)t * k + j];
        Vec<T, V> a;
        a.load(o + (size_t)r * d + c);
#pragma unroll
        for (int i = 0; i < V; ++i) acc.v[i] = fmaf(g, a.v[i], acc.v[i]);
      }
      acc.store(y + (size_t)t * d + c);
    }
  }
}

// per padded row r: do[r] = g_r * dy[token(r)] (0 for padding rows); dgate[pair(r)] = <dy[token], o[r]>
template <typename T, int V>
__global__ void __launch_bounds__(kRowThreads)
combine_bwd_kernel(const T* __restrict__ dy, const T* __restrict__ o, const int32_t* __restrict__ prow_token,
                   const float* __restrict__ prow_gate, const int32_t* __restrict__ prow_pair,
                   const int32_t* __restrict__ n_mtiles, int d, T* __restrict__ dop, float* __restrict__ dgate) {
  pdl_launch_dependents();
  pdl_wait();
  __shared__ float red[kRowThreads / 32];
  const int rows = n_mtiles[1];
  for (int r = blockIdx.x; r < rows; r += gridDim.x) {
    const int t = prow_token[r];
    const float g = t >= 0 ? prow_gate[r] : 0.f;
    float dot = 0.f;
    for (int c = threadIdx.x * V; c < d; c += kRowThreads * V) {
      Vec<T, V> a, b;
      if (t >= 0) {
        a.load(dy + (size_t)t * d + c);
        b.load(o + (size_t)r * d + c);
#pragma unroll
        for (int i = 0; i < V; ++i) { dot = fmaf(a.v[i], b.v[i], dot); a.v[i] *= g; }
      } else {
        a.zero();
      }
      a.store(dop + (size_t)r * d + c);
    }
    if (t >= 0) {  // block-uniform branch
#pragma unroll
      for (int s = 16; s > 0; s >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, s);
      if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = dot;
      __syncthreads();
      if (threadIdx.x == 0) {
        float s = 0.f;
        for (int w = 0; w < kRowThreads / 32; ++w) s += red[w];
        dgate[prow_pair[r]] = s;
      }
      __syncthreads();
    }
  }
}

// do[r] = g_r * dy[token(r)] only (0 for padding rows): B1 without the <dy, o> dot, for the path whose dgate comes out of the
// DH epilogue (umma_gemm.cu)
template <typename T, int V>
__global__ void __launch_bounds__(kRowThreads)
scale_rows_kernel(const T* __restrict__ dy, const int32_t* __restrict__ prow_token, const float* __restrict__ prow_gate,
                  const int32_t* __restrict__ n_mtiles, int d, T* __restrict__ dop) {
  pdl_launch_dependents();
  pdl_wait();
  const int rows = n_mtiles[1];
  for (int r = blockIdx.x; r < rows; r += gridDim.x) {
    const int t = prow_token[r];
    const float g = t >= 0 ? prow_gate[r] : 0.f;
    for (int c = threadIdx.x * V; c < d; c += kRowThreads * V) {
      Vec<T, V> a;
      if (t >= 0) {
        a.load(dy + (size_t)t * d + c);
#pragma unroll
        for (int i = 0; i < V; ++i) a.v[i] *= g;
      } else {
        a.zero();
      }
      a.store(dop + (size_t)r * d + c);
    }
  }
}

// Gate rule + gate function backward (row B6): dz[t,:] from dgate[t,:].  One warp per token.
// DZ = float (row stride E) or bf16 (row stride ldz >= E, padding columns zeroed: K-operand of the tensor-core router backward)
template <typename DZ>
__global__ void gate_bwd_kernel(const float* __restrict__ probs, const int32_t* __restrict__ topk_idx,
                                const float* __restrict__ gate, const int32_t* __restrict__ pair_prow,
                                const float* __restrict__ dgate, const float* __restrict__ dgate_part, int n_parts, int T_, int E,
                                int k, int gate_fn, int gate_rule, float inv_tau, DZ* __restrict__ dz, int ldz) {
  pdl_launch_dependents();
  pdl_wait();
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= T_) return;
  const int t = warp;
  // lanes j < k own selected pair j
  int e = -1;
  bool kept = false;
  float dg = 0.f, g = 0.f, p = 0.f;
  if (lane < k) {
    e = topk_idx[(size_t)t * k + lane];
    const int pr = pair_prow[(size_t)t * k + lane];
    kept = pr >= 0;
    g = gate[(size_t)t * k + lane];
    p = probs[(size_t)t * E + e];
    if (kept && dgate_part) {   // <dy, o> = <dh, h> / g with dh = g dy W_down: partial sums from the DH epilogue, fixed order
      const int np = n_parts < 0 ? -n_parts : n_parts;   // n_parts < 0: the partials are <dy W_down, h> itself, not scaled by g
      float sacc = 0.f;
      for (int i = 0; i < np; ++i) sacc += dgate_part[(size_t)pr * np + i];
      dg = n_parts < 0 ? sacc : g != 0.f ? sacc / g : 0.f;
    } else {
      dg = kept ? dgate[(size_t)t * k + lane] : 0.f;
    }
  }
  float dp = 0.f;  // dL/dp of the expert this lane owns
  if (gate_rule == FOMOE_DROP_ONLY) {
    dp = kept ? dg : 0.f;
  } else {
    const bool in_norm = lane < k && (gate_rule == FOMOE_RENORM_TOPK || kept);
    float ssum = in_norm ? p : 0.f, dgg = kept ? dg * g : 0.f;
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
      ssum += __shfl_xor_sync(0xffffffffu, ssum, s);
      dgg += __shfl_xor_sync(0xffffffffu, dgg, s);
    }
    dp = (in_norm && ssum > 0.f) ? ((kept ? dg : 0.f) - dgg) / ssum : 0.f;
  }
  if (gate_fn == FOMOE_GATE_SIGMOID) {
    for (int ee = lane; ee < ldz; ee += 32) dz[(size_t)t * ldz + ee] = from_f32<DZ>(0.f);
    __syncwarp();
    if (lane < k) dz[(size_t)t * ldz + e] = from_f32<DZ>(dp * p * (1.f - p) * inv_tau);
  } else {
    float pd = lane < k ? p * dp : 0.f;
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) pd += __shfl_xor_sync(0xffffffffu, pd, s);
    for (int ee = lane; ee < ldz; ee += 32)
      dz[(size_t)t * ldz + ee] = from_f32<DZ>(ee < E ? probs[(size_t)t * E + ee] * (0.f - pd) * inv_tau : 0.f);
    __syncwarp();
    if (lane < k) dz[(size_t)t * ldz + e] = from_f32<DZ>(p * (dp - pd) * inv_tau);
  }
}

// dx[t] = sum_{j ascending} dxp[pair_prow[t,j]] + dx_sh[t] + dx_r[t]   (router term as fp32 or in the element type)
template <typename T, int V>
__global__ void __launch_bounds__(kRowThreads)
dx_sum_kernel(const T* __restrict__ dxp, const T* __restrict__ dx_sh, const float* __restrict__ dx_r, const T* __restrict__ dx_r_t,
              const int32_t* __restrict__ pair_prow, int T_, int d, int k, int rpb, T* __restrict__ dx) {
  pdl_launch_dependents();
  pdl_wait();
  const int tpr = kRowThreads / rpb, sub = threadIdx.x / tpr, c0 = (threadIdx.x % tpr) * V;   // (as in combine_kernel)
  for (int t = blockIdx.x * rpb + sub; t < T_; t += gridDim.x * rpb) {
    for (int c = c0; c < d; c += tpr * V) {
      Vec<T, V> acc;
      if (dx_sh) acc.load(dx_sh + (size_t)t * d + c); else acc.zero();
      for (int j = 0; j < k; ++j) {
        const int r = pair_prow[(size_t)t * k + j];
        if (r < 0) continue;
        Vec<T, V> a;
        a.load(dxp + (size_t)r * d + c);
#pragma unroll
        for (int i = 0; i < V; ++i) acc.v[i] += a.v[i];
      }
      if (dx_r) {
#pragma unroll
        for (int i = 0; i < V; ++i) acc.v[i] += dx_r[(size_t)t * d + c + i];
      }
      if (dx_r_t) {
        Vec<T, V> a;
        a.load(dx_r_t + (size_t)t * d + c);
#pragma unroll
        for (int i = 0; i < V; ++i) acc.v[i] += a.v[i];
      }
      acc.store(dx + (size_t)t * d + c);
    }
  }
}

// token rows per CTA of combine / dx_sum: the largest power of two (<= 8) whose rows' vector chunks fit the CTA's threads
// (d = 512 bf16: 64 chunks -> 2 rows; on P1 dx_sum 25 -> 20 us, combine 16 -> 14 us); 1 once d / V > kRowThreads / 2
static int rows_per_block(int d, int V) {
  const int n = (d + V - 1) / V;
  int r = 1;
  while (r < 8 && n * r * 2 <= kRowThreads) r *= 2;
  return r;
}

// dispatch on dtype and on whether rows are 16-byte vectorisable
#define ROWS_DISPATCH(c, CALL)                                              \
  do {                                                                      \
    if ((c).dtype == FOMOE_BF16) {                                          \
      using T = __nv_bfloat16;                                              \
      if ((c).d_model % 8 == 0) { constexpr int V = 8; CALL; } else { constexpr int V = 1; CALL; } \
    } else {                                                                \
      using T = float;                                                      \
      if ((c).d_model % 4 == 0) { constexpr int V = 4; CALL; } else { constexpr int V = 1; CALL; } \
    }                                                                       \
  } while (0)

int launch_gather_rows(const fomoe_config& c, const void* x, const RouteWs& ws, void* xp, cudaStream_t st) {
  ROWS_DISPATCH(c, FOMOE_CUDA_OK(launch_pdl(gather_rows_kernel<T, V>, row_grid(ws.R_cap, c.d_model), kRowThreads, 0, st, (const T*)x, ws.prow_token,
                                            ws.n_mtiles, c.d_model, (T*)xp)));
  FOMOE_LAUNCH_OK("gather_rows_kernel");
  return FOMOE_OK;
}

int launch_combine(const fomoe_config& c, const fomoe_route_state& r, const RouteWs& ws, const void* o, const void* y_sh,
                   void* y, cudaStream_t st) {
  if (c.T == 0) return FOMOE_OK;
  ROWS_DISPATCH(c, const int rpb = rows_per_block(c.d_model, V);
                FOMOE_CUDA_OK(launch_pdl(combine_kernel<T, V>, row_grid(ceil_div(c.T, rpb), c.d_model * rpb), kRowThreads, 0, st, (const T*)o,
                                         (const T*)y_sh, r.gate, ws.pair_prow, c.T, c.d_model, c.top_k, rpb, (T*)y)));
  FOMOE_LAUNCH_OK("combine_kernel");
  return FOMOE_OK;
}

int launch_combine_bwd(const fomoe_config& c, const void* dy, const void* o, const RouteWs& ws, void* dop, float* dgate,
                       cudaStream_t st) {
  // dgate is written for every kept pair and read (gate_bwd_kernel) for kept pairs only: no clearing needed
  ROWS_DISPATCH(c, FOMOE_CUDA_OK(launch_pdl(combine_bwd_kernel<T, V>, row_grid(ws.R_cap, c.d_model), kRowThreads, 0, st, (const T*)dy, (const T*)o,
                                            ws.prow_token, ws.prow_gate, ws.prow_pair, ws.n_mtiles, c.d_model, (T*)dop, dgate)));
  FOMOE_LAUNCH_OK("combine_bwd_kernel");
  return FOMOE_OK;
}

int launch_scale_rows(const fomoe_config& c, const void* dy, const RouteWs& ws, void* dop, cudaStream_t st) {
  ROWS_DISPATCH(c, FOMOE_CUDA_OK(launch_pdl(scale_rows_kernel<T, V>, row_grid(ws.R_cap, c.d_model), kRowThreads, 0, st, (const T*)dy, ws.prow_token,
                                            ws.prow_gate, ws.n_mtiles, c.d_model, (T*)dop)));
  FOMOE_LAUNCH_OK("scale_rows_kernel");
  return FOMOE_OK;
}

int launch_gate_bwd(const fomoe_config& c, const fomoe_route_state& r, const RouteWs& ws, const float* dgate, const float* dgate_part,
                    int n_parts, float* dz, void* dz_bf, int ldz_bf, cudaStream_t st) {
  if (c.T == 0) return FOMOE_OK;
  if (dz_bf)
    FOMOE_CUDA_OK(launch_pdl(gate_bwd_kernel<__nv_bfloat16>, ceil_div(c.T, 8), 256, 0, st, r.probs, r.topk_idx, r.gate, ws.pair_prow, dgate,
                             dgate_part, n_parts, c.T, c.E, c.top_k, c.gate_fn, c.gate_rule, 1.0f / c.temperature, (__nv_bfloat16*)dz_bf,
                             ldz_bf));
  else
    FOMOE_CUDA_OK(launch_pdl(gate_bwd_kernel<float>, ceil_div(c.T, 8), 256, 0, st, r.probs, r.topk_idx, r.gate, ws.pair_prow, dgate,
                             dgate_part, n_parts, c.T, c.E, c.top_k, c.gate_fn, c.gate_rule, 1.0f / c.temperature, dz, c.E));
  FOMOE_LAUNCH_OK("gate_bwd_kernel");
  return FOMOE_OK;
}

int launch_dx_sum(const fomoe_config& c, const RouteWs& ws, const void* dxp, const void* dx_sh, const float* dx_r, const void* dx_r_t,
                  void* dx, cudaStream_t st) {
  if (c.T == 0) return FOMOE_OK;
  ROWS_DISPATCH(c, const int rpb = rows_per_block(c.d_model, V);
                FOMOE_CUDA_OK(launch_pdl(dx_sum_kernel<T, V>, row_grid(ceil_div(c.T, rpb), c.d_model * rpb), kRowThreads, 0, st, (const T*)dxp,
                                         (const T*)dx_sh, dx_r, (const T*)dx_r_t, ws.pair_prow, c.T, c.d_model, c.top_k, rpb, (T*)dx)));
  FOMOE_LAUNCH_OK("dx_sum_kernel");
  return FOMOE_OK;
}

}  // namespace fomoe
