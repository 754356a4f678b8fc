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
  for (int i = 0; i < (int)(blockDim.x >> 5); ++i) s += red[i];   // same order in every thread
  return s;
}

// 16-byte vector access: VN elements of T as fp32 (bf16: 8, fp32: 4)
template <typename T> struct VecN { static constexpr int n = 16 / sizeof(T); };
template <typename T> __device__ __forceinline__ void ldv(const T* p, float (&v)[VecN<T>::n]);
template <> __device__ __forceinline__ void ldv<float>(const float* p, float (&v)[4]) {
  const float4 r = *reinterpret_cast<const float4*>(p);
  v[0] = r.x; v[1] = r.y; v[2] = r.z; v[3] = r.w;
}
template <> __device__ __forceinline__ void ldv<__nv_bfloat16>(const __nv_bfloat16* p, float (&v)[8]) {
  const uint4 r = *reinterpret_cast<const uint4*>(p);
  const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&r);
#pragma unroll
  for (int i = 0; i < 4; ++i) { const float2 f = __bfloat1622float2(h[i]); v[2 * i] = f.x; v[2 * i + 1] = f.y; }
}
template <typename T> __device__ __forceinline__ void stv(T* p, const float (&v)[VecN<T>::n]);
template <> __device__ __forceinline__ void stv<float>(float* p, const float (&v)[4]) {
  *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}
template <> __device__ __forceinline__ void stv<__nv_bfloat16>(__nv_bfloat16* p, const float (&v)[8]) {
  uint4 r;
  __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&r);
#pragma unroll
  for (int i = 0; i < 4; ++i) h[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]);
  *reinterpret_cast<uint4*>(p) = r;
}

template <typename T>
__global__ void __launch_bounds__(kLnThreads)
periln_fwd_kernel(const T* __restrict__ x, const float* __restrict__ gamma, const float* __restrict__ beta, const T* __restrict__ residual,
                  float alpha, float eps, int T_, int d, T* __restrict__ out, float* __restrict__ stats) {
  extern __shared__ float row[];   // [d]
  __shared__ float red[kLnThreads / 32];
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const T* xr = x + (size_t)t * d;
    constexpr int VN = VecN<T>::n;
    const bool vec = d % VN == 0;
    float s = 0.f;
    if (vec) {
      for (int c = threadIdx.x * VN; c < d; c += kLnThreads * VN) {
        float v[VN];
        ldv<T>(xr + c, v);
#pragma unroll
        for (int i = 0; i < VN; ++i) { row[c + i] = v[i]; s += v[i]; }
      }
    } else {
      for (int c = threadIdx.x; c < d; c += kLnThreads) { const float v = to_f32(xr[c]); row[c] = v; s += v; }
    }
    const float mean = block_sum(s, red) / (float)d;
    float q = 0.f;
    for (int c = threadIdx.x; c < d; c += kLnThreads) { const float v = row[c] - mean; q += v * v; }
    const float rstd = rsqrtf(block_sum(q, red) / (float)d + eps);
    if (threadIdx.x == 0) { stats[2 * (size_t)t] = mean; stats[2 * (size_t)t + 1] = rstd; }
    if (vec) {
      for (int c = threadIdx.x * VN; c < d; c += kLnThreads * VN) {
        float v[VN], r[VN];
        if (residual) ldv<T>(residual + (size_t)t * d + c, r);
#pragma unroll
        for (int i = 0; i < VN; ++i) {
          v[i] = alpha * (gamma[c + i] * ((row[c + i] - mean) * rstd) + beta[c + i]);
          if (residual) v[i] += r[i];
        }
        stv<T>(out + (size_t)t * d + c, v);
      }
    } else {
      for (int c = threadIdx.x; c < d; c += kLnThreads) {
        float v = alpha * (gamma[c] * ((row[c] - mean) * rstd) + beta[c]);
        if (residual) v += to_f32(residual[(size_t)t * d + c]);
        out[(size_t)t * d + c] = from_f32<T>(v);
      }
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
  __syncthreads();   // the accumulation below maps columns to threads differently (16-byte vectors)
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const float mean = stats[2 * (size_t)t], rstd = stats[2 * (size_t)t + 1];
    float s1 = 0.f, s2 = 0.f;
    constexpr int VN = VecN<T>::n;
    const bool vec = d % VN == 0;   // a thread owns the same columns in every pass and for every token either way
    if (vec) {
      for (int c = threadIdx.x * VN; c < d; c += kLnThreads * VN) {
        float go[VN], xv[VN];
        ldv<T>(dout + (size_t)t * d + c, go);
        ldv<T>(x + (size_t)t * d + c, xv);
#pragma unroll
        for (int i = 0; i < VN; ++i) {
          const float g = alpha * go[i], h = (xv[i] - mean) * rstd, dh = g * gamma[c + i];
          xh[c + i] = h; dxh[c + i] = dh;
          ag[c + i] += g * h;
          ab[c + i] += g;
          s1 += dh; s2 += dh * h;
        }
      }
    } else {
      for (int c = threadIdx.x; c < d; c += kLnThreads) {
        const float go = alpha * to_f32(dout[(size_t)t * d + c]);
        const float h = (to_f32(x[(size_t)t * d + c]) - mean) * rstd;
        const float dh = go * gamma[c];
        xh[c] = h; dxh[c] = dh;
        ag[c] += go * h;               // each column is owned by one thread: no atomics, fixed token order
        ab[c] += go;
        s1 += dh; s2 += dh * h;
      }
    }
    const float m1 = block_sum(s1, red) / (float)d;
    const float m2 = block_sum(s2, red) / (float)d;
    if (vec) {
      for (int c = threadIdx.x * VN; c < d; c += kLnThreads * VN) {
        float v[VN], r[VN];
        if (dresidual) ldv<T>(dresidual + (size_t)t * d + c, r);
#pragma unroll
        for (int i = 0; i < VN; ++i) {
          v[i] = rstd * (dxh[c + i] - m1 - xh[c + i] * m2);
          if (dresidual) v[i] += r[i];
        }
        stv<T>(dx + (size_t)t * d + c, v);
      }
    } else {
      for (int c = threadIdx.x; c < d; c += kLnThreads) {
        float v = rstd * (dxh[c] - m1 - xh[c] * m2);
        if (dresidual) v += to_f32(dresidual[(size_t)t * d + c]);
        dx[(size_t)t * d + c] = from_f32<T>(v);
      }
    }
  }
  __syncthreads();
  for (int c = threadIdx.x; c < d; c += kLnThreads) {
    partials[((size_t)blockIdx.x * 2) * d + c] = ag[c];
    partials[((size_t)blockIdx.x * 2 + 1) * d + c] = ab[c];
  }
}

// ---- register-resident variants (d a multiple of the vector width, at most NV vectors per thread): the row never touches
// shared memory, gamma and the dgamma / dbeta accumulators live in registers across the CTA's tokens ----
template <typename T, int NV>
__global__ void __launch_bounds__(kLnThreads)
periln_fwd_reg_kernel(const T* __restrict__ x, const float* __restrict__ gamma, const float* __restrict__ beta, const T* __restrict__ residual,
                      float alpha, float eps, int T_, int d, T* __restrict__ out, float* __restrict__ stats) {
  constexpr int VN = VecN<T>::n;
  __shared__ float red[kLnThreads / 32];
  float g[NV][VN], b[NV][VN];
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
#pragma unroll
    for (int i = 0; i < VN; ++i) { g[j][i] = c < d ? gamma[c + i] : 0.f; b[j][i] = c < d ? beta[c + i] : 0.f; }
  }
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const size_t base = (size_t)t * d;
    float v[NV][VN], r[NV][VN];
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
        ldv<T>(x + base + c, v[j]);
        if (residual) ldv<T>(residual + base + c, r[j]);
#pragma unroll
        for (int i = 0; i < VN; ++i) s += v[j][i];
      }
    }
    const float mean = block_sum(s, red) / (float)d;
    float q = 0.f;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
#pragma unroll
        for (int i = 0; i < VN; ++i) { v[j][i] -= mean; q += v[j][i] * v[j][i]; }
      }
    }
    const float rstd = rsqrtf(block_sum(q, red) / (float)d + eps);
    if (threadIdx.x == 0) { stats[2 * (size_t)t] = mean; stats[2 * (size_t)t + 1] = rstd; }
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
#pragma unroll
        for (int i = 0; i < VN; ++i) {
          v[j][i] = alpha * (g[j][i] * (v[j][i] * rstd) + b[j][i]);
          if (residual) v[j][i] += r[j][i];
        }
        stv<T>(out + base + c, v[j]);
      }
    }
  }
}

template <typename T, int NV>
__global__ void __launch_bounds__(kLnThreads)
periln_bwd_reg_kernel(const T* __restrict__ dout, const T* __restrict__ x, const float* __restrict__ stats, const float* __restrict__ gamma,
                      float alpha, const T* __restrict__ dresidual, int T_, int d, T* __restrict__ dx, float* __restrict__ partials) {
  constexpr int VN = VecN<T>::n;
  __shared__ float red[kLnThreads / 32];
  float g[NV][VN], ag[NV][VN], ab[NV][VN];
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
#pragma unroll
    for (int i = 0; i < VN; ++i) { g[j][i] = c < d ? gamma[c + i] : 0.f; ag[j][i] = 0.f; ab[j][i] = 0.f; }
  }
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const size_t base = (size_t)t * d;
    const float mean = stats[2 * (size_t)t], rstd = stats[2 * (size_t)t + 1];
    float dh[NV][VN], h[NV][VN], r[NV][VN];
    float s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
        ldv<T>(dout + base + c, dh[j]);
        ldv<T>(x + base + c, h[j]);
        if (dresidual) ldv<T>(dresidual + base + c, r[j]);
#pragma unroll
        for (int i = 0; i < VN; ++i) {
          const float go = alpha * dh[j][i];
          h[j][i] = (h[j][i] - mean) * rstd;
          ag[j][i] += go * h[j][i];          // fixed token order per CTA
          ab[j][i] += go;
          dh[j][i] = go * g[j][i];
          s1 += dh[j][i];
          s2 += dh[j][i] * h[j][i];
        }
      }
    }
    const float m1 = block_sum(s1, red) / (float)d;
    const float m2 = block_sum(s2, red) / (float)d;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
#pragma unroll
        for (int i = 0; i < VN; ++i) {
          dh[j][i] = rstd * (dh[j][i] - m1 - h[j][i] * m2);
          if (dresidual) dh[j][i] += r[j][i];
        }
        stv<T>(dx + base + c, dh[j]);
      }
    }
  }
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
    if (c < d) {
#pragma unroll
      for (int i = 0; i < VN; ++i) {
        partials[((size_t)blockIdx.x * 2) * d + c + i] = ag[j][i];
        partials[((size_t)blockIdx.x * 2 + 1) * d + c + i] = ab[j][i];
      }
    }
  }
}

// dgamma / dbeta = sum over the CTAs' partials, in a fixed order: a CTA owns 32 columns; 32 row groups each sum every 32nd
// partial (loads batched 4 deep), then group 0 adds the 32 group sums in order
__global__ void __launch_bounds__(1024)
periln_reduce_kernel(const float* __restrict__ partials, int n_blk, int d, float* __restrict__ dgamma, float* __restrict__ dbeta) {
  __shared__ float sg[32][33], sb[32][33];
  const int col = threadIdx.x & 31, grp = threadIdx.x >> 5, c = blockIdx.x * 32 + col;
  float g = 0.f, b = 0.f;
  if (c < d) {
    int i = grp;
    for (; i + 96 < n_blk; i += 128) {
      float gv[4], bv[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        gv[u] = partials[((size_t)(i + 32 * u) * 2) * d + c];
        bv[u] = partials[((size_t)(i + 32 * u) * 2 + 1) * d + c];
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) { g += gv[u]; b += bv[u]; }
    }
    for (; i < n_blk; i += 32) { g += partials[((size_t)i * 2) * d + c]; b += partials[((size_t)i * 2 + 1) * d + c]; }
  }
  sg[grp][col] = g;
  sb[grp][col] = b;
  __syncthreads();
  if (grp == 0 && c < d) {
    float tg = 0.f, tb = 0.f;
#pragma unroll
    for (int k = 0; k < 32; ++k) { tg += sg[k][col]; tb += sb[k][col]; }
    dgamma[c] = tg;
    dbeta[c] = tb;
  }
}

}  // namespace

int periln_blocks(int T) { int g = num_sms() * 8; if (g > T) g = T; return g < 1 ? 1 : g; }

// threads per CTA and vectors per thread needed to hold one row in registers; nv = 0: use the shared-memory kernels
template <typename T> static void reg_shape(int d, int& threads, int& nv) {
  const int vn = VecN<T>::n;
  threads = kLnThreads;
  nv = 0;
  if (d % vn) return;
  const int vecs = d / vn;
  threads = vecs <= 256 ? 128 : 256;            // narrow rows: more CTAs per SM instead of idle lanes
  const int need = ceil_div(vecs, threads);
  nv = need <= 1 ? 1 : need <= 2 ? 2 : need <= 4 ? 4 : 0;
  if (nv == 0) threads = kLnThreads;
}

template <typename T>
static int periln_fwd_t(int Tn, int d, const void* x, const float* gamma, const float* beta, float eps, const void* residual, float alpha,
                        void* out, float* stats, cudaStream_t st) {
  int threads, nv;
  reg_shape<T>(d, threads, nv);
  const int grid = Tn < num_sms() * 16 ? Tn : num_sms() * 16;
#define LN_FWD(NV) periln_fwd_reg_kernel<T, NV><<<grid, threads, 0, st>>>((const T*)x, gamma, beta, (const T*)residual, alpha, eps, Tn, d, (T*)out, stats)
  if (nv == 1) LN_FWD(1);
  else if (nv == 2) LN_FWD(2);
  else if (nv == 4) LN_FWD(4);
  else {
    const size_t smem = sizeof(float) * (size_t)d;
    FOMOE_CUDA_OK(cudaFuncSetAttribute(periln_fwd_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    periln_fwd_kernel<T><<<grid, kLnThreads, smem, st>>>((const T*)x, gamma, beta, (const T*)residual, alpha, eps, Tn, d, (T*)out, stats);
  }
#undef LN_FWD
  FOMOE_LAUNCH_OK("periln_fwd_kernel");
  return FOMOE_OK;
}

int launch_periln_fwd(int T, int d, int dtype, const void* x, const float* gamma, const float* beta, float eps, const void* residual,
                      float alpha, void* out, float* stats, cudaStream_t st) {
  if (T == 0) return FOMOE_OK;
  return dtype == FOMOE_BF16 ? periln_fwd_t<__nv_bfloat16>(T, d, x, gamma, beta, eps, residual, alpha, out, stats, st)
                             : periln_fwd_t<float>(T, d, x, gamma, beta, eps, residual, alpha, out, stats, st);
}

template <typename T>
static int periln_bwd_t(int Tn, int d, int nb, const void* dout, const void* x, const float* stats, const float* gamma, float alpha,
                        const void* dresidual, void* dx, float* partials, cudaStream_t st) {
  int threads, nv;
  reg_shape<T>(d, threads, nv);
#define LN_BWD(NV) periln_bwd_reg_kernel<T, NV><<<nb, threads, 0, st>>>((const T*)dout, (const T*)x, stats, gamma, alpha, (const T*)dresidual, Tn, d, (T*)dx, partials)
  if (nv == 1) LN_BWD(1);
  else if (nv == 2) LN_BWD(2);
  else if (nv == 4) LN_BWD(4);
  else {
    const size_t smem = sizeof(float) * 4 * (size_t)d;
    FOMOE_CUDA_OK(cudaFuncSetAttribute(periln_bwd_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    periln_bwd_kernel<T><<<nb, kLnThreads, smem, st>>>((const T*)dout, (const T*)x, stats, gamma, alpha, (const T*)dresidual, Tn, d, (T*)dx, partials);
  }
#undef LN_BWD
  FOMOE_LAUNCH_OK("periln_bwd_kernel");
  return FOMOE_OK;
}

int launch_periln_bwd(int T, int d, int dtype, const void* dout, const void* x, const float* stats, const float* gamma, float alpha,
                      const void* dresidual, void* dx, float* dgamma, float* dbeta, float* partials, cudaStream_t st) {
  const int nb = periln_blocks(T);
  if (T > 0) {
    int rc = dtype == FOMOE_BF16 ? periln_bwd_t<__nv_bfloat16>(T, d, nb, dout, x, stats, gamma, alpha, dresidual, dx, partials, st)
                                 : periln_bwd_t<float>(T, d, nb, dout, x, stats, gamma, alpha, dresidual, dx, partials, st);
    if (rc != FOMOE_OK) return rc;
  }
  periln_reduce_kernel<<<ceil_div(d, 32), 1024, 0, st>>>(partials, T > 0 ? nb : 0, d, dgamma, dbeta);
  FOMOE_LAUNCH_OK("periln_reduce_kernel");
  return FOMOE_OK;
}

}  // namespace fomoe
