// Peripheral LayerNorm either side of the MoE block:  x_{l+1} = x_l + alpha LN(F(LN(x_l)))
// (Eq. 15; depth multiplier PAPER.md:601 Fig. 12).  Two streaming row kernels, one CTA per token row at a time:
//   periln_fwd : out = [residual +] alpha (gamma xhat + beta), saves (mean, rstd)       — pre-LN (no residual) and post-LN + residual
//   periln_bwd : dx = [dresidual +] rstd (dxhat - mean(dxhat) - xhat mean(dxhat xhat)), dxhat = alpha dout gamma;
//                per-CTA partial dgamma / dbeta, summed by a second kernel in a fixed order (run-to-run identical)
// The row is staged once in shared memory (fp32), so mean and the centred variance are computed exactly as LayerNorm
// defines them and global memory is read once.  Bound: HBM.
#include "common.cuh"

namespace fomoe {
namespace {

constexpr int kLnThreads = 256;

__device__ __forceinline__ float block_sum(float v, float* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  __syncthreads();                 // red may still be read from the previous call
  if (l == 0) red[w] = v;
  __syncthreads();
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < kLnThreads / 32; ++i) s += red[i];   // same order in every thread
  return s;
}

template <typename T>
__global__ void __launch_bounds__(kLnThreads)
periln_fwd_kernel(const T* __restrict__ x, const float* __restrict__ gamma, const float* __restrict__ beta, const T* __restrict__ residual,
                  float alpha, float eps, int T_, int d, T* __restrict__ out, float* __restrict__ stats) {
  extern __shared__ float row[];   // [d]
  __shared__ float red[kLnThreads / 32];
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const T* xr = x + (size_t)t * d;
    float s = 0.f;
    for (int c = threadIdx.x; c < d; c += kLnThreads) { const float v = to_f32(xr[c]); row[c] = v; s += v; }
    const float mean = block_sum(s, red) / (float)d;
    float q = 0.f;
    for (int c = threadIdx.x; c < d; c += kLnThreads) { const float v = row[c] - mean; q += v * v; }
    const float rstd = rsqrtf(block_sum(q, red) / (float)d + eps);
    if (threadIdx.x == 0) { stats[2 * (size_t)t] = mean; stats[2 * (size_t)t + 1] = rstd; }
    for (int c = threadIdx.x; c < d; c += kLnThreads) {
      float v = alpha * (gamma[c] * ((row[c] - mean) * rstd) + beta[c]);
      if (residual) v += to_f32(residual[(size_t)t * d + c]);
      out[(size_t)t * d + c] = from_f32<T>(v);
    }
    __syncthreads();
  }
}

template <typename T>
__global__ void __launch_bounds__(kLnThreads)
periln_bwd_kernel(const T* __restrict__ dout, const T* __restrict__ x, const float* __restrict__ stats, const float* __restrict__ gamma,
                  float alpha, const T* __restrict__ dresidual, int T_, int d, T* __restrict__ dx, float* __restrict__ partials) {
  extern __shared__ float sm[];    // xhat [d] | dxhat [d] | dgamma acc [d] | dbeta acc [d]
  float *xh = sm, *dxh = sm + d, *ag = sm + 2 * d, *ab = sm + 3 * d;
  __shared__ float red[kLnThreads / 32];
  for (int c = threadIdx.x; c < d; c += kLnThreads) { ag[c] = 0.f; ab[c] = 0.f; }
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const float mean = stats[2 * (size_t)t], rstd = stats[2 * (size_t)t + 1];
    float s1 = 0.f, s2 = 0.f;
    for (int c = threadIdx.x; c < d; c += kLnThreads) {
      const float go = alpha * to_f32(dout[(size_t)t * d + c]);
      const float h = (to_f32(x[(size_t)t * d + c]) - mean) * rstd;
      const float dh = go * gamma[c];
      xh[c] = h; dxh[c] = dh;
      ag[c] += go * h;               // each column is owned by one thread: no atomics, fixed token order
      ab[c] += go;
      s1 += dh; s2 += dh * h;
    }
    const float m1 = block_sum(s1, red) / (float)d;
    const float m2 = block_sum(s2, red) / (float)d;
    for (int c = threadIdx.x; c < d; c += kLnThreads) {
      float v = rstd * (dxh[c] - m1 - xh[c] * m2);
      if (dresidual) v += to_f32(dresidual[(size_t)t * d + c]);
      dx[(size_t)t * d + c] = from_f32<T>(v);
    }
  }
  for (int c = threadIdx.x; c < d; c += kLnThreads) {
    partials[((size_t)blockIdx.x * 2) * d + c] = ag[c];
    partials[((size_t)blockIdx.x * 2 + 1) * d + c] = ab[c];
  }
}

__global__ void periln_reduce_kernel(const float* __restrict__ partials, int n_blk, int d, float* __restrict__ dgamma, float* __restrict__ dbeta) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= d) return;
  float g = 0.f, b = 0.f;
  for (int i = 0; i < n_blk; ++i) { g += partials[((size_t)i * 2) * d + c]; b += partials[((size_t)i * 2 + 1) * d + c]; }
  dgamma[c] = g;
  dbeta[c] = b;
}

}  // namespace

int periln_blocks(int T) { int g = 148 * 4; if (g > T) g = T; return g < 1 ? 1 : g; }

int launch_periln_fwd(int T, int d, int dtype, const void* x, const float* gamma, const float* beta, float eps, const void* residual,
                      float alpha, void* out, float* stats, cudaStream_t st) {
  if (T == 0) return FOMOE_OK;
  const size_t smem = sizeof(float) * (size_t)d;
  const int grid = T < 148 * 8 ? T : 148 * 8;
  if (dtype == FOMOE_BF16) {
    using E = __nv_bfloat16;
    FOMOE_CUDA_OK(cudaFuncSetAttribute(periln_fwd_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    periln_fwd_kernel<E><<<grid, kLnThreads, smem, st>>>((const E*)x, gamma, beta, (const E*)residual, alpha, eps, T, d, (E*)out, stats);
  } else {
    FOMOE_CUDA_OK(cudaFuncSetAttribute(periln_fwd_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    periln_fwd_kernel<float><<<grid, kLnThreads, smem, st>>>((const float*)x, gamma, beta, (const float*)residual, alpha, eps, T, d,
                                                             (float*)out, stats);
  }
  FOMOE_LAUNCH_OK("periln_fwd_kernel");
  return FOMOE_OK;
}

int launch_periln_bwd(int T, int d, int dtype, const void* dout, const void* x, const float* stats, const float* gamma, float alpha,
                      const void* dresidual, void* dx, float* dgamma, float* dbeta, float* partials, cudaStream_t st) {
  const int nb = periln_blocks(T);
  if (T > 0) {
    const size_t smem = sizeof(float) * 4 * (size_t)d;
    if (dtype == FOMOE_BF16) {
      using E = __nv_bfloat16;
      FOMOE_CUDA_OK(cudaFuncSetAttribute(periln_bwd_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      periln_bwd_kernel<E><<<nb, kLnThreads, smem, st>>>((const E*)dout, (const E*)x, stats, gamma, alpha, (const E*)dresidual, T, d, (E*)dx,
                                                         partials);
    } else {
      FOMOE_CUDA_OK(cudaFuncSetAttribute(periln_bwd_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      periln_bwd_kernel<float><<<nb, kLnThreads, smem, st>>>((const float*)dout, (const float*)x, stats, gamma, alpha,
                                                             (const float*)dresidual, T, d, (float*)dx, partials);
    }
    FOMOE_LAUNCH_OK("periln_bwd_kernel");
  }
  periln_reduce_kernel<<<ceil_div(d, 256), 256, 0, st>>>(partials, T > 0 ? nb : 0, d, dgamma, dbeta);
  FOMOE_LAUNCH_OK("periln_reduce_kernel");
  return FOMOE_OK;
}

}  // namespace fomoe
