// Peripheral LayerNorm either side of the MoE block:  x_{l+1} = x_l + alpha LN(F(LN(x_l)))
// (Eq. 15; depth multiplier PAPER.md:601 Fig. 12).  Two streaming row kernels, one CTA per token row at a time:
//   periln_fwd : out = [residual +] alpha (gamma xhat + beta), saves (mean, rstd)       — pre-LN (no residual) and post-LN + residual
//   periln_bwd : dx = [dresidual +] rstd (dxhat - mean(dxhat) - xhat mean(dxhat xhat)), dxhat = alpha dout gamma;
//                per-CTA partial dgamma / dbeta, summed by a second kernel in a fixed order (run-to-run identical)
// Three forms of each: *_ring_kernel (rows prefetched by cp.async.bulk into a shared-memory ring, gamma / beta and the
// accumulators in registers: the default for rows of at most two 16-byte vectors per thread), *_reg_kernel (row held in
// registers, more CTAs per SM) and the general kernel that stages the row in shared memory as fp32.  Mean and the centred
// variance are computed exactly as LayerNorm defines them and global memory is read once.  Bound: HBM.
#include "common.cuh"
#include "umma_ptx.cuh"
#include <stdio.h>
#include <stdlib.h>

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

// two independent sums through the same tree as block_sum (so each equals what block_sum would return), one barrier pair
__device__ __forceinline__ void block_sum2(float& a, float& b, float* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (int)(blockDim.x >> 5);
  __syncthreads();
  if (l == 0) { red[w] = a; red[nw + w] = b; }
  __syncthreads();
  float sa = 0.f, sb = 0.f;
#pragma unroll
  for (int i = 0; i < nw; ++i) { sa += red[i]; sb += red[nw + i]; }
  a = sa; b = sb;
}

// The element formulas, with every rounding spelled out (no compiler-chosen FMA contraction): the stand-alone kernels and the
// forms fused into combine / dx_sum (below) must produce the same bits.
__device__ __forceinline__ float ln_out(float centred, float rstd, float g, float b, float alpha, bool has_res, float res) {
  const float t = __fmaf_rn(g, __fmul_rn(centred, rstd), b);
  return has_res ? __fmaf_rn(alpha, t, res) : __fmul_rn(alpha, t);
}
__device__ __forceinline__ float ln_dx(float rstd, float dxhat, float m1, float xhat, float m2, bool has_res, float res) {
  const float t = __fmul_rn(rstd, __fmaf_rn(-xhat, m2, __fsub_rn(dxhat, m1)));
  return has_res ? __fadd_rn(t, res) : t;
}
// accumulates one element into (dgamma, dbeta, sum dxhat, sum dxhat xhat); returns dxhat = go * gamma
__device__ __forceinline__ float ln_bwd_acc(float go, float xhat, float g, float& ag, float& ab, float& s1, float& s2) {
  ag = __fmaf_rn(go, xhat, ag);
  ab = __fadd_rn(ab, go);
  const float dxh = __fmul_rn(go, g);
  s1 = __fadd_rn(s1, dxh);
  s2 = __fmaf_rn(dxh, xhat, s2);
  return dxh;
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
// a 16-byte vector kept as loaded (bf16: 8 values in 4 registers) and widened when used: the register count decides how many
// rows an SM keeps in flight
template <typename T> __device__ __forceinline__ void unpack(const uint4& r, float (&v)[VecN<T>::n]);
template <> __device__ __forceinline__ void unpack<float>(const uint4& r, float (&v)[4]) {
  v[0] = __uint_as_float(r.x); v[1] = __uint_as_float(r.y); v[2] = __uint_as_float(r.z); v[3] = __uint_as_float(r.w);
}
template <> __device__ __forceinline__ void unpack<__nv_bfloat16>(const uint4& r, float (&v)[8]) {
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
        for (int i = 0; i < VN; ++i) v[i] = ln_out(row[c + i] - mean, rstd, gamma[c + i], beta[c + i], alpha, residual != nullptr, residual ? r[i] : 0.f);
        stv<T>(out + (size_t)t * d + c, v);
      }
    } else {
      for (int c = threadIdx.x; c < d; c += kLnThreads) {
        const float v = ln_out(row[c] - mean, rstd, gamma[c], beta[c], alpha, residual != nullptr, residual ? to_f32(residual[(size_t)t * d + c]) : 0.f);
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
          const float g = __fmul_rn(alpha, go[i]), h = __fmul_rn(xv[i] - mean, rstd);
          xh[c + i] = h;
          dxh[c + i] = ln_bwd_acc(g, h, gamma[c + i], ag[c + i], ab[c + i], s1, s2);
        }
      }
    } else {
      for (int c = threadIdx.x; c < d; c += kLnThreads) {
        const float go = __fmul_rn(alpha, to_f32(dout[(size_t)t * d + c]));
        const float h = __fmul_rn(to_f32(x[(size_t)t * d + c]) - mean, rstd);
        xh[c] = h;
        dxh[c] = ln_bwd_acc(go, h, gamma[c], ag[c], ab[c], s1, s2);   // each column is owned by one thread: no atomics, fixed token order
      }
    }
    const float m1 = block_sum(s1, red) / (float)d;
    const float m2 = block_sum(s2, red) / (float)d;
    if (vec) {
      for (int c = threadIdx.x * VN; c < d; c += kLnThreads * VN) {
        float v[VN], r[VN];
        if (dresidual) ldv<T>(dresidual + (size_t)t * d + c, r);
#pragma unroll
        for (int i = 0; i < VN; ++i) v[i] = ln_dx(rstd, dxh[c + i], m1, xh[c + i], m2, dresidual != nullptr, dresidual ? r[i] : 0.f);
        stv<T>(dx + (size_t)t * d + c, v);
      }
    } else {
      for (int c = threadIdx.x; c < d; c += kLnThreads) {
        const float v = ln_dx(rstd, dxh[c], m1, xh[c], m2, dresidual != nullptr, dresidual ? to_f32(dresidual[(size_t)t * d + c]) : 0.f);
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
// gamma / beta are re-read per token (16-byte loads, L1-resident) instead of living in registers: the register count decides how
// many rows an SM keeps in flight, and these kernels are bound by exactly that
template <typename T, int VN> __device__ __forceinline__ void ld_param(const float* p, float (&v)[VN]) {
  ldv<float>(p, *reinterpret_cast<float(*)[4]>(&v[0]));
  if constexpr (VN == 8) ldv<float>(p + 4, *reinterpret_cast<float(*)[4]>(&v[4]));
}

// The row is held as loaded (bf16: 8 values in 4 registers) and widened each time it is used: with <= 40 registers per thread
// six CTAs are resident per SM, and the number of rows in flight per SM is what bounds this kernel.
template <typename T, int NV, bool RES>   // RES: a residual row is read and added (post-LN); without it two more CTAs fit per SM
__global__ void __launch_bounds__(kLnThreads, NV <= 2 ? (RES ? 5 : 6) : 2)
periln_fwd_reg_kernel(const T* __restrict__ x, const float* __restrict__ gamma, const float* __restrict__ beta, const T* __restrict__ residual,
                      float alpha, float eps, int T_, int d, T* __restrict__ out, float* __restrict__ stats) {
  constexpr int VN = VecN<T>::n;
  __shared__ float red[kLnThreads / 32];
  pdl_launch_dependents();
  pdl_wait();
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const size_t base = (size_t)t * d;
    uint4 xr[NV], rr[NV];
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      xr[j] = make_uint4(0u, 0u, 0u, 0u);
      rr[j] = make_uint4(0u, 0u, 0u, 0u);
      if (c < d) {
        xr[j] = *reinterpret_cast<const uint4*>(x + base + c);
        if (RES) rr[j] = *reinterpret_cast<const uint4*>(residual + base + c);
      }
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
        float v[VN];
        unpack<T>(xr[j], v);
#pragma unroll
        for (int i = 0; i < VN; ++i) s += v[i];
      }
    }
    const float mean = block_sum(s, red) / (float)d;
    float q = 0.f;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
        float v[VN];
        unpack<T>(xr[j], v);
#pragma unroll
        for (int i = 0; i < VN; ++i) { v[i] -= mean; q += v[i] * v[i]; }
      }
    }
    const float rstd = rsqrtf(block_sum(q, red) / (float)d + eps);
    if (threadIdx.x == 0) { stats[2 * (size_t)t] = mean; stats[2 * (size_t)t + 1] = rstd; }
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
        float g[VN], b[VN], v[VN], r[VN];
        ld_param<T, VN>(gamma + c, g);
        ld_param<T, VN>(beta + c, b);
        unpack<T>(xr[j], v);
        unpack<T>(rr[j], r);
#pragma unroll
        for (int i = 0; i < VN; ++i) v[i] = ln_out(v[i] - mean, rstd, g[i], b[i], alpha, RES, r[i]);
        stv<T>(out + base + c, v);
      }
    }
  }
}

// The same kernel with the row loads taken off the critical path: thread 0 keeps a ring of kRingStages rows per CTA filled with
// bulk copies (cp.async.bulk, completion on an mbarrier), kRingStages rows ahead of the row being normalised, so the bytes an
// SM has in flight no longer depend on how many CTAs' registers fit.  Every thread then reads exactly the vectors it would
// have loaded from global memory, and the arithmetic below that point is periln_fwd_reg_kernel's, statement for statement
// (same bits).  Rows of d * sizeof(T) bytes, 16-byte multiples.
constexpr int kRingStages = 3;
__device__ __forceinline__ void bulk_row_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
template <typename T, int NV, bool RES>
__global__ void __launch_bounds__(kLnThreads, 3)
periln_fwd_ring_kernel(const T* __restrict__ x, const float* __restrict__ gamma, const float* __restrict__ beta, const T* __restrict__ residual,
                       float alpha, float eps, int T_, int d, T* __restrict__ out, float* __restrict__ stats) {
  constexpr int VN = VecN<T>::n;
  extern __shared__ __align__(128) uint8_t ring[];   // [kRingStages][x row | residual row]
  __shared__ float red[kLnThreads / 32];
  __shared__ __align__(8) uint64_t full[kRingStages];
  const uint32_t row_bytes = (uint32_t)d * sizeof(T), stage_bytes = row_bytes * (RES ? 2 : 1);
  const uint32_t ring0 = smem_u32(ring), full0 = smem_u32(full);
  if (threadIdx.x == 0) {
    for (int s = 0; s < kRingStages; ++s) mbar_init(full0 + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  pdl_launch_dependents();
  pdl_wait();
  auto issue = [&](int t, int s) {   // thread 0: row t into stage s
    mbar_expect_tx(full0 + 8 * s, stage_bytes);
    bulk_row_load(ring0 + s * stage_bytes, x + (size_t)t * d, row_bytes, full0 + 8 * s);
    if (RES) bulk_row_load(ring0 + s * stage_bytes + row_bytes, residual + (size_t)t * d, row_bytes, full0 + 8 * s);
  };
  if (threadIdx.x == 0)
    for (int s = 0; s < kRingStages; ++s) {
      const long t = (long)blockIdx.x + (long)s * gridDim.x;
      if (t < T_) issue((int)t, s);
    }
  // with the loads prefetched, occupancy no longer decides the bytes in flight: gamma / beta live in registers for the whole
  // kernel and the row is widened to fp32 once (the register-resident kernel re-reads 4 bytes of gamma / beta per byte of row
  // from L1 and widens the row three times: ncu shows it bound by issue slots and the L1 pipe, not by DRAM)
  float g[NV][VN], b[NV][VN];
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
#pragma unroll
    for (int i = 0; i < VN; ++i) { g[j][i] = 0.f; b[j][i] = 0.f; }
    if (c < d) { ld_param<T, VN>(gamma + c, g[j]); ld_param<T, VN>(beta + c, b[j]); }
  }
  int stage = 0;
  uint32_t phase = 0;
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const size_t base = (size_t)t * d;
    float v[NV][VN];
    uint4 rr[NV];
    mbar_wait(full0 + 8 * stage, phase);
    const uint32_t srow = ring0 + stage * stage_bytes;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      uint4 xr = make_uint4(0u, 0u, 0u, 0u);
      rr[j] = make_uint4(0u, 0u, 0u, 0u);
      if (c < d) {
        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(xr.x), "=r"(xr.y), "=r"(xr.z), "=r"(xr.w)
                     : "r"(srow + c * (uint32_t)sizeof(T)) : "memory");
        if (RES)
          asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(rr[j].x), "=r"(rr[j].y), "=r"(rr[j].z), "=r"(rr[j].w)
                       : "r"(srow + row_bytes + c * (uint32_t)sizeof(T)) : "memory");
      }
      unpack<T>(xr, v[j]);
    }
    __syncthreads();   // every thread has its vectors: the stage can be refilled
    if (threadIdx.x == 0) {
      const long tn = (long)t + (long)kRingStages * gridDim.x;
      if (tn < T_) issue((int)tn, stage);
    }
    if (++stage == kRingStages) { stage = 0; phase ^= 1; }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
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
        float r[VN], o[VN];
        unpack<T>(rr[j], r);
#pragma unroll
        for (int i = 0; i < VN; ++i) o[i] = ln_out(v[j][i], rstd, g[j][i], b[j][i], alpha, RES, r[i]);
        stv<T>(out + base + c, o);
      }
    }
  }
}

// Rows held as loaded (see periln_fwd_reg_kernel).  The dgamma / dbeta accumulators live in shared memory when the row is at
// most two vectors per thread (each thread reads and writes only its own columns: no conflicts, no atomics, fixed token
// order), which brings the kernel from 80-127 registers to <= 64 and from 2-3 resident CTAs per SM to 4.
template <typename T, int NV>
__global__ void __launch_bounds__(kLnThreads, NV <= 2 ? 4 : 1)
periln_bwd_reg_kernel(const T* __restrict__ dout, const T* __restrict__ x, const float* __restrict__ stats, const float* __restrict__ gamma,
                      float alpha, const T* __restrict__ dresidual, int T_, int d, T* __restrict__ dx, float* __restrict__ partials) {
  constexpr int VN = VecN<T>::n;
  constexpr bool kSmemAcc = NV <= 2;
  extern __shared__ float acc_sm[];          // kSmemAcc: [2][d] dgamma | dbeta accumulators of this CTA
  __shared__ float red[2 * (kLnThreads / 32)];
  pdl_launch_dependents();
  pdl_wait();
  float ag[kSmemAcc ? 1 : NV][VN], ab[kSmemAcc ? 1 : NV][VN];
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
#pragma unroll
    for (int i = 0; i < VN; ++i) {
      if (kSmemAcc) { if (c < d) { acc_sm[c + i] = 0.f; acc_sm[d + c + i] = 0.f; } }
      else { ag[j][i] = 0.f; ab[j][i] = 0.f; }
    }
  }
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const size_t base = (size_t)t * d;
    const float mean = stats[2 * (size_t)t], rstd = stats[2 * (size_t)t + 1];
    uint4 gr[NV], xr[NV], rr[NV];
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      gr[j] = xr[j] = rr[j] = make_uint4(0u, 0u, 0u, 0u);
      if (c < d) {
        gr[j] = *reinterpret_cast<const uint4*>(dout + base + c);
        xr[j] = *reinterpret_cast<const uint4*>(x + base + c);
        if (dresidual) rr[j] = *reinterpret_cast<const uint4*>(dresidual + base + c);
      }
    }
    float s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
        float g[VN], go[VN], h[VN], a_g[VN], a_b[VN];
        ld_param<T, VN>(gamma + c, g);
        unpack<T>(gr[j], go);
        unpack<T>(xr[j], h);
        if (kSmemAcc) { ld_param<T, VN>(acc_sm + c, a_g); ld_param<T, VN>(acc_sm + d + c, a_b); }
#pragma unroll
        for (int i = 0; i < VN; ++i) {
          const float gi = __fmul_rn(alpha, go[i]);
          const float hi = __fmul_rn(h[i] - mean, rstd);
          if (kSmemAcc) ln_bwd_acc(gi, hi, g[i], a_g[i], a_b[i], s1, s2);   // fixed token order per CTA
          else ln_bwd_acc(gi, hi, g[i], ag[j][i], ab[j][i], s1, s2);
        }
        if (kSmemAcc) {
#pragma unroll
          for (int v4 = 0; v4 < VN / 4; ++v4) {
            *reinterpret_cast<float4*>(acc_sm + c + 4 * v4) = make_float4(a_g[4 * v4], a_g[4 * v4 + 1], a_g[4 * v4 + 2], a_g[4 * v4 + 3]);
            *reinterpret_cast<float4*>(acc_sm + d + c + 4 * v4) = make_float4(a_b[4 * v4], a_b[4 * v4 + 1], a_b[4 * v4 + 2], a_b[4 * v4 + 3]);
          }
        }
      }
    }
    block_sum2(s1, s2, red);
    const float m1 = s1 / (float)d, m2 = s2 / (float)d;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
        float g[VN], go[VN], h[VN], r[VN];
        ld_param<T, VN>(gamma + c, g);
        unpack<T>(gr[j], go);
        unpack<T>(xr[j], h);
        unpack<T>(rr[j], r);
#pragma unroll
        for (int i = 0; i < VN; ++i) {
          const float dxh = __fmul_rn(__fmul_rn(alpha, go[i]), g[i]);          // the same roundings as in ln_bwd_acc
          const float hi = __fmul_rn(h[i] - mean, rstd);
          go[i] = ln_dx(rstd, dxh, m1, hi, m2, dresidual != nullptr, r[i]);
        }
        stv<T>(dx + base + c, go);
      }
    }
  }
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
    if (c < d) {
#pragma unroll
      for (int i = 0; i < VN; ++i) {
        partials[((size_t)blockIdx.x * 2) * d + c + i] = kSmemAcc ? acc_sm[c + i] : ag[j][i];
        partials[((size_t)blockIdx.x * 2 + 1) * d + c + i] = kSmemAcc ? acc_sm[d + c + i] : ab[j][i];
      }
    }
  }
}

// The backward with its rows prefetched through the same kind of ring (dout row | x row | dresidual row per stage) and, since
// occupancy no longer matters, gamma and the dgamma / dbeta accumulators in registers for the whole kernel (the register kernel
// above reads and writes 16 bytes of shared-memory accumulators and re-reads 8 bytes of gamma per byte of row).  Same grid,
// same token order per CTA and the same element formulas as periln_bwd_reg_kernel: same bits, partials included.
template <typename T, int NV, bool RES>
__global__ void __launch_bounds__(kLnThreads, 2)
periln_bwd_ring_kernel(const T* __restrict__ dout, const T* __restrict__ x, const float* __restrict__ stats, const float* __restrict__ gamma,
                       float alpha, const T* __restrict__ dresidual, int T_, int d, T* __restrict__ dx, float* __restrict__ partials) {
  constexpr int VN = VecN<T>::n;
  constexpr int kRows = RES ? 3 : 2;
  extern __shared__ __align__(128) uint8_t ring[];
  __shared__ float red[2 * (kLnThreads / 32)];
  __shared__ __align__(8) uint64_t full[kRingStages];
  const uint32_t row_bytes = (uint32_t)d * sizeof(T), stage_bytes = row_bytes * kRows;
  const uint32_t ring0 = smem_u32(ring), full0 = smem_u32(full);
  if (threadIdx.x == 0) {
    for (int s = 0; s < kRingStages; ++s) mbar_init(full0 + 8 * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  pdl_launch_dependents();
  pdl_wait();
  auto issue = [&](int t, int s) {
    mbar_expect_tx(full0 + 8 * s, stage_bytes);
    bulk_row_load(ring0 + s * stage_bytes, dout + (size_t)t * d, row_bytes, full0 + 8 * s);
    bulk_row_load(ring0 + s * stage_bytes + row_bytes, x + (size_t)t * d, row_bytes, full0 + 8 * s);
    if (RES) bulk_row_load(ring0 + s * stage_bytes + 2 * row_bytes, dresidual + (size_t)t * d, row_bytes, full0 + 8 * s);
  };
  if (threadIdx.x == 0)
    for (int s = 0; s < kRingStages; ++s) {
      const long t = (long)blockIdx.x + (long)s * gridDim.x;
      if (t < T_) issue((int)t, s);
    }
  float g[NV][VN], ag[NV][VN], ab[NV][VN];
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
#pragma unroll
    for (int i = 0; i < VN; ++i) { g[j][i] = 0.f; ag[j][i] = 0.f; ab[j][i] = 0.f; }
    if (c < d) ld_param<T, VN>(gamma + c, g[j]);
  }
  int stage = 0;
  uint32_t phase = 0;
  float2 st_cur = blockIdx.x < T_ ? *reinterpret_cast<const float2*>(stats + 2 * (size_t)blockIdx.x) : make_float2(0.f, 0.f);
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const size_t base = (size_t)t * d;
    const float mean = st_cur.x, rstd = st_cur.y;
    if ((long)t + gridDim.x < T_) st_cur = *reinterpret_cast<const float2*>(stats + 2 * ((size_t)t + gridDim.x));   // next row's, early
    float gi[NV][VN], hi[NV][VN];
    uint4 rr[NV];
    mbar_wait(full0 + 8 * stage, phase);
    const uint32_t srow = ring0 + stage * stage_bytes;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      uint4 gr = make_uint4(0u, 0u, 0u, 0u), xr = make_uint4(0u, 0u, 0u, 0u);
      rr[j] = make_uint4(0u, 0u, 0u, 0u);
      if (c < d) {
        const uint32_t a = srow + c * (uint32_t)sizeof(T);
        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(gr.x), "=r"(gr.y), "=r"(gr.z), "=r"(gr.w) : "r"(a) : "memory");
        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(xr.x), "=r"(xr.y), "=r"(xr.z), "=r"(xr.w) : "r"(a + row_bytes) : "memory");
        if (RES)
          asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(rr[j].x), "=r"(rr[j].y), "=r"(rr[j].z), "=r"(rr[j].w)
                       : "r"(a + 2 * row_bytes) : "memory");
      }
      unpack<T>(gr, gi[j]);
      unpack<T>(xr, hi[j]);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      const long tn = (long)t + (long)kRingStages * gridDim.x;
      if (tn < T_) issue((int)tn, stage);
    }
    if (++stage == kRingStages) { stage = 0; phase ^= 1; }
    float s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
#pragma unroll
        for (int i = 0; i < VN; ++i) {
          gi[j][i] = __fmul_rn(alpha, gi[j][i]);
          hi[j][i] = __fmul_rn(hi[j][i] - mean, rstd);
          ln_bwd_acc(gi[j][i], hi[j][i], g[j][i], ag[j][i], ab[j][i], s1, s2);   // fixed token order per CTA
        }
      }
    }
    block_sum2(s1, s2, red);
    const float m1 = s1 / (float)d, m2 = s2 / (float)d;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * (int)blockDim.x + threadIdx.x) * VN;
      if (c < d) {
        float r[VN], o[VN];
        unpack<T>(rr[j], r);
#pragma unroll
        for (int i = 0; i < VN; ++i) {
          const float dxh = __fmul_rn(gi[j][i], g[j][i]);          // the same roundings as in ln_bwd_acc
          o[i] = ln_dx(rstd, dxh, m1, hi[j][i], m2, RES, r[i]);
        }
        stv<T>(dx + base + c, o);
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

// ---- fused into the MoE layer's own row kernels (SURVEY.md §8(f) row 3 as written: "post-LN + depth multiplier + residual
// fused into combine"; the pre-LN backward + residual into the dx scatter-sum).  A CTA holds a whole token row in registers
// either way, so the LayerNorm statistics cost two block reductions and no extra pass over [T, d].  The sums run in exactly
// the order of combine_kernel / dx_sum_kernel (rows.cu) and the LayerNorm is applied to the value ROUNDED to the storage type,
// so the fused path is bit-identical to combine -> fomoe_periln_fwd and dx_sum -> fomoe_periln_bwd. ----

// y[t] = sum_j gate[t,j] o[pair_prow[t,j]] (+ y_sh[t])  (saved: the post-LN backward needs it);
// out[t] = residual[t] + alpha (gamma xhat(y[t]) + beta); stats[t] = (mean, rstd)
template <typename T, int NV, int THREADS>
__global__ void __launch_bounds__(THREADS, NV <= 2 ? 1024 / THREADS : 1)
combine_periln_kernel(const T* __restrict__ o, const T* __restrict__ y_sh, const float* __restrict__ gate, const int32_t* __restrict__ pair_prow,
                      int T_, int d, int k, T* __restrict__ y, const float* __restrict__ gamma, const float* __restrict__ beta,
                      const T* __restrict__ residual, float alpha, float eps, T* __restrict__ out, float* __restrict__ stats) {
  constexpr int VN = VecN<T>::n;
  __shared__ float red[THREADS / 32];
  pdl_launch_dependents();
  pdl_wait();
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const size_t base = (size_t)t * d;
    float v[NV][VN];
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * THREADS + threadIdx.x) * VN;
      if (c < d && y_sh) ldv<T>(y_sh + base + c, v[j]);
      else {
#pragma unroll
        for (int i = 0; i < VN; ++i) v[j][i] = 0.f;
      }
    }
    for (int jj = 0; jj < k; ++jj) {          // ascending j: the order of combine_kernel
      const int r = pair_prow[(size_t)t * k + jj];
      if (r < 0) continue;
      const float g = gate[(size_t)t * k + jj];
#pragma unroll
      for (int j = 0; j < NV; ++j) {
        const int c = (j * THREADS + threadIdx.x) * VN;
        if (c < d) {
          float a[VN];
          ldv<T>(o + (size_t)r * d + c, a);
#pragma unroll
          for (int i = 0; i < VN; ++i) v[j][i] = fmaf(g, a[i], v[j][i]);
        }
      }
    }
    float rres[NV][VN];                        // residual row: requested before the reductions
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * THREADS + threadIdx.x) * VN;
      if (c < d) ldv<T>(residual + base + c, rres[j]);
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * THREADS + threadIdx.x) * VN;
      if (c < d) {
        stv<T>(y + base + c, v[j]);
#pragma unroll
        for (int i = 0; i < VN; ++i) { v[j][i] = to_f32(from_f32<T>(v[j][i])); s += v[j][i]; }   // LayerNorm of what was stored
      }
    }
    const float mean = block_sum(s, red) / (float)d;
    float q = 0.f;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * THREADS + threadIdx.x) * VN;
      if (c < d) {
#pragma unroll
        for (int i = 0; i < VN; ++i) { v[j][i] -= mean; q += v[j][i] * v[j][i]; }
      }
    }
    const float rstd = rsqrtf(block_sum(q, red) / (float)d + eps);
    if (threadIdx.x == 0) { stats[2 * (size_t)t] = mean; stats[2 * (size_t)t + 1] = rstd; }
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * THREADS + threadIdx.x) * VN;
      if (c < d) {
        float gm[VN], bt[VN];
        ldv<float>(gamma + c, *reinterpret_cast<float(*)[4]>(&gm[0]));
        ldv<float>(beta + c, *reinterpret_cast<float(*)[4]>(&bt[0]));
        if constexpr (VN == 8) {
          ldv<float>(gamma + c + 4, *reinterpret_cast<float(*)[4]>(&gm[4]));
          ldv<float>(beta + c + 4, *reinterpret_cast<float(*)[4]>(&bt[4]));
        }
#pragma unroll
        for (int i = 0; i < VN; ++i) v[j][i] = ln_out(v[j][i], rstd, gm[i], bt[i], alpha, true, rres[j][i]);
        stv<T>(out + base + c, v[j]);
      }
    }
  }
}

// dxn[t] = sum_j dxp[pair_prow[t,j]] + dx_sh[t] + dx_r[t]  (gradient w.r.t. the pre-LN output; never stored);
// dx[t] = dresidual[t] + LN backward of dxn[t] at (x_raw[t], stats[t], gamma); per-CTA partial dgamma / dbeta
template <typename T, int NV, int THREADS>
__global__ void __launch_bounds__(THREADS, NV <= 2 ? 768 / THREADS : 1)
dx_sum_periln_kernel(const T* __restrict__ dxp, const T* __restrict__ dx_sh, const float* __restrict__ dx_r, const T* __restrict__ dx_r_t,
                     const int32_t* __restrict__ pair_prow, int T_, int d, int k, const T* __restrict__ x_raw, const float* __restrict__ stats,
                     const float* __restrict__ gamma, const T* __restrict__ dresidual, T* __restrict__ dx, float* __restrict__ partials) {
  constexpr int VN = VecN<T>::n;
  constexpr bool kSmemAcc = NV <= 2;          // (as in periln_bwd_reg_kernel: accumulators in shared memory, rows held as loaded)
  extern __shared__ float acc_sm[];
  __shared__ float red[2 * (THREADS / 32)];
  pdl_launch_dependents();
  pdl_wait();
  float ag[kSmemAcc ? 1 : NV][VN], ab[kSmemAcc ? 1 : NV][VN];
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const int c = (j * THREADS + threadIdx.x) * VN;
#pragma unroll
    for (int i = 0; i < VN; ++i) {
      if (kSmemAcc) { if (c < d) { acc_sm[c + i] = 0.f; acc_sm[d + c + i] = 0.f; } }
      else { ag[j][i] = 0.f; ab[j][i] = 0.f; }
    }
  }
  for (int t = blockIdx.x; t < T_; t += gridDim.x) {
    const size_t base = (size_t)t * d;
    float dh[NV][VN];
    uint4 xr[NV], rr[NV];                      // block input row and residual-branch gradient: requested early, used last
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * THREADS + threadIdx.x) * VN;
      if (c < d && dx_sh) ldv<T>(dx_sh + base + c, dh[j]);
      else {
#pragma unroll
        for (int i = 0; i < VN; ++i) dh[j][i] = 0.f;
      }
      xr[j] = rr[j] = make_uint4(0u, 0u, 0u, 0u);
      if (c < d) {
        xr[j] = *reinterpret_cast<const uint4*>(x_raw + base + c);
        if (dresidual) rr[j] = *reinterpret_cast<const uint4*>(dresidual + base + c);
      }
    }
    for (int jj = 0; jj < k; ++jj) {          // the order of dx_sum_kernel
      const int r = pair_prow[(size_t)t * k + jj];
      if (r < 0) continue;
#pragma unroll
      for (int j = 0; j < NV; ++j) {
        const int c = (j * THREADS + threadIdx.x) * VN;
        if (c < d) {
          float a[VN];
          ldv<T>(dxp + (size_t)r * d + c, a);
#pragma unroll
          for (int i = 0; i < VN; ++i) dh[j][i] += a[i];
        }
      }
    }
    const float mean = stats[2 * (size_t)t], rstd = stats[2 * (size_t)t + 1];
    float s1 = 0.f, s2 = 0.f;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * THREADS + threadIdx.x) * VN;
      if (c < d) {
        if (dx_r) {
#pragma unroll
          for (int i = 0; i < VN; ++i) dh[j][i] += dx_r[base + c + i];
        }
        if (dx_r_t) {
          float a[VN];
          ldv<T>(dx_r_t + base + c, a);
#pragma unroll
          for (int i = 0; i < VN; ++i) dh[j][i] += a[i];
        }
        float gm[VN], h[VN], a_g[VN], a_b[VN];
        ld_param<T, VN>(gamma + c, gm);
        unpack<T>(xr[j], h);
        if (kSmemAcc) { ld_param<T, VN>(acc_sm + c, a_g); ld_param<T, VN>(acc_sm + d + c, a_b); }
#pragma unroll
        for (int i = 0; i < VN; ++i) {
          const float go = to_f32(from_f32<T>(dh[j][i]));      // what dx_sum_kernel would have stored (alpha = 1)
          const float hi = __fmul_rn(h[i] - mean, rstd);
          if (kSmemAcc) dh[j][i] = ln_bwd_acc(go, hi, gm[i], a_g[i], a_b[i], s1, s2);   // fixed token order per CTA
          else dh[j][i] = ln_bwd_acc(go, hi, gm[i], ag[j][i], ab[j][i], s1, s2);
        }
        if (kSmemAcc) {
#pragma unroll
          for (int v4 = 0; v4 < VN / 4; ++v4) {
            *reinterpret_cast<float4*>(acc_sm + c + 4 * v4) = make_float4(a_g[4 * v4], a_g[4 * v4 + 1], a_g[4 * v4 + 2], a_g[4 * v4 + 3]);
            *reinterpret_cast<float4*>(acc_sm + d + c + 4 * v4) = make_float4(a_b[4 * v4], a_b[4 * v4 + 1], a_b[4 * v4 + 2], a_b[4 * v4 + 3]);
          }
        }
      }
    }
    block_sum2(s1, s2, red);
    const float m1 = s1 / (float)d, m2 = s2 / (float)d;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      const int c = (j * THREADS + threadIdx.x) * VN;
      if (c < d) {
        float h[VN], r[VN];
        unpack<T>(xr[j], h);
        unpack<T>(rr[j], r);
#pragma unroll
        for (int i = 0; i < VN; ++i) dh[j][i] = ln_dx(rstd, dh[j][i], m1, __fmul_rn(h[i] - mean, rstd), m2, dresidual != nullptr, r[i]);
        stv<T>(dx + base + c, dh[j]);
      }
    }
  }
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const int c = (j * THREADS + threadIdx.x) * VN;
    if (c < d) {
#pragma unroll
      for (int i = 0; i < VN; ++i) {
        partials[((size_t)blockIdx.x * 2) * d + c + i] = kSmemAcc ? acc_sm[c + i] : ag[j][i];
        partials[((size_t)blockIdx.x * 2 + 1) * d + c + i] = kSmemAcc ? acc_sm[d + c + i] : ab[j][i];
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

// CTAs of the backward kernels = partial dgamma / dbeta sums: 4 per SM is one wave of the register-resident and of the fused
// kernels (4 CTAs resident) and two waves of the ring kernel (2 resident); every CTA costs 2 d floats of partial-sum traffic
int periln_blocks(int T) { int g = num_sms() * 4; if (g > T) g = T; return g < 1 ? 1 : g; }

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
  const int grid_reg = Tn < num_sms() * 32 ? Tn : num_sms() * 32;
  const int grid = Tn < num_sms() * 16 ? Tn : num_sms() * 16;
  static const int ring_mode = [] { const char* e = getenv("FOMOE_LN_RING"); return e ? atoi(e) : 1; }();   // FOMOE_LN_RING=0: the register-resident kernels
  if (ring_mode && nv >= 1 && nv <= 2 && ((size_t)d * sizeof(T)) % 16 == 0) {
    const size_t smem = (size_t)kRingStages * d * sizeof(T) * (residual ? 2 : 1);
    const int ctas = threads == kLnThreads ? 3 : 6;
    const int grid_ring = Tn < num_sms() * ctas ? Tn : num_sms() * ctas;
#define LN_RING(NV, RES)                                                                                                            \
    do {                                                                                                                          \
      static PerDeviceOnce attr;                                                                                                  \
      if (attr.need()) { FOMOE_CUDA_OK(cudaFuncSetAttribute(periln_fwd_ring_kernel<T, NV, RES>, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024)); attr.set(); } \
      FOMOE_CUDA_OK(launch_pdl(periln_fwd_ring_kernel<T, NV, RES>, grid_ring, threads, smem, st, (const T*)x, gamma, beta, (const T*)residual, \
                               alpha, eps, Tn, d, (T*)out, stats));                                                               \
    } while (0)
    if (smem <= 96 * 1024) {
      if (nv == 1) { if (residual) LN_RING(1, true); else LN_RING(1, false); }
      else { if (residual) LN_RING(2, true); else LN_RING(2, false); }
      FOMOE_LAUNCH_OK("periln_fwd_ring_kernel");
      return FOMOE_OK;
    }
#undef LN_RING
  }
#define LN_FWD(NV)                                                                                                                  \
  do {                                                                                                                            \
    if (residual) FOMOE_CUDA_OK(launch_pdl(periln_fwd_reg_kernel<T, NV, true>, grid_reg, threads, 0, st, (const T*)x, gamma, beta,      \
                                           (const T*)residual, alpha, eps, Tn, d, (T*)out, stats));                                \
    else FOMOE_CUDA_OK(launch_pdl(periln_fwd_reg_kernel<T, NV, false>, grid_reg, threads, 0, st, (const T*)x, gamma, beta,              \
                                  (const T*)residual, alpha, eps, Tn, d, (T*)out, stats));                                         \
  } while (0)
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
  static const int ring_mode = [] { const char* e = getenv("FOMOE_LN_RING"); return e ? atoi(e) : 1; }();   // FOMOE_LN_RING=0: the register-resident kernels
  if (ring_mode && nv >= 1 && nv <= 2 && ((size_t)d * sizeof(T)) % 16 == 0) {
    const size_t smem = (size_t)kRingStages * d * sizeof(T) * (dresidual ? 3 : 2);
#define LN_BRING(NV, RES)                                                                                                          \
    do {                                                                                                                          \
      static PerDeviceOnce attr;                                                                                                  \
      if (attr.need()) { FOMOE_CUDA_OK(cudaFuncSetAttribute(periln_bwd_ring_kernel<T, NV, RES>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024)); attr.set(); } \
      FOMOE_CUDA_OK(launch_pdl(periln_bwd_ring_kernel<T, NV, RES>, nb, threads, smem, st, (const T*)dout, (const T*)x, stats, gamma, alpha, \
                               (const T*)dresidual, Tn, d, (T*)dx, partials));                                                    \
    } while (0)
    if (smem <= 100 * 1024) {
      if (nv == 1) { if (dresidual) LN_BRING(1, true); else LN_BRING(1, false); }
      else { if (dresidual) LN_BRING(2, true); else LN_BRING(2, false); }
      FOMOE_LAUNCH_OK("periln_bwd_ring_kernel");
      return FOMOE_OK;
    }
#undef LN_BRING
  }
#define LN_BWD(NV) FOMOE_CUDA_OK(launch_pdl(periln_bwd_reg_kernel<T, NV>, nb, threads, (NV <= 2 ? sizeof(float) * 2 * (size_t)d : 0), st, (const T*)dout, (const T*)x, stats, gamma, alpha, (const T*)dresidual, Tn, d, (T*)dx, partials))
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

// ---- launchers of the fused forms; return FOMOE_ERR_UNSUPPORTED when the row does not fit the register-resident shape
// (the caller then runs the unfused sequence) ----
bool periln_fused_supported(const fomoe_config& c) {
  int threads, nv;
  if (c.dtype == FOMOE_BF16) reg_shape<__nv_bfloat16>(c.d_model, threads, nv); else reg_shape<float>(c.d_model, threads, nv);
  return nv != 0;
}

template <typename T>
static int combine_periln_t(const fomoe_config& c, const fomoe_route_state& r, const RouteWs& ws, const void* o, const void* y_sh, void* y,
                            const fomoe_periln_post& ln, cudaStream_t st) {
  int threads, nv;
  reg_shape<T>(c.d_model, threads, nv);
  const int grid = c.T < num_sms() * 16 ? c.T : num_sms() * 16;
#define CB(NV, TH) FOMOE_CUDA_OK(launch_pdl(combine_periln_kernel<T, NV, TH>, grid, TH, 0, st, (const T*)o, (const T*)y_sh, (const float*)r.gate, \
    (const int32_t*)ws.pair_prow, c.T, c.d_model, c.top_k, (T*)y, ln.gamma, ln.beta, (const T*)ln.residual, ln.alpha, ln.eps, (T*)ln.out, ln.stats))
  if (threads == 128) { if (nv == 1) CB(1, 128); else if (nv == 2) CB(2, 128); else return FOMOE_ERR_UNSUPPORTED; }
  else { if (nv == 2) CB(2, 256); else if (nv == 4) CB(4, 256); else return FOMOE_ERR_UNSUPPORTED; }
#undef CB
  FOMOE_LAUNCH_OK("combine_periln_kernel");
  return FOMOE_OK;
}

int launch_combine_periln(const fomoe_config& c, const fomoe_route_state& r, const RouteWs& ws, const void* o, const void* y_sh, void* y,
                          const fomoe_periln_post& ln, cudaStream_t st) {
  if (c.T == 0) return FOMOE_OK;
  return c.dtype == FOMOE_BF16 ? combine_periln_t<__nv_bfloat16>(c, r, ws, o, y_sh, y, ln, st) : combine_periln_t<float>(c, r, ws, o, y_sh, y, ln, st);
}

template <typename T>
static int dx_sum_periln_t(const fomoe_config& c, const RouteWs& ws, const void* dxp, const void* dx_sh, const float* dx_r, const void* dx_r_t,
                           const fomoe_periln_pre_bwd& ln, void* dx, int nb, cudaStream_t st) {
  int threads, nv;
  reg_shape<T>(c.d_model, threads, nv);
#define DB(NV, TH) FOMOE_CUDA_OK(launch_pdl(dx_sum_periln_kernel<T, NV, TH>, nb, TH, (NV <= 2 ? sizeof(float) * 2 * (size_t)c.d_model : 0), st, (const T*)dxp, (const T*)dx_sh, dx_r, (const T*)dx_r_t, \
    (const int32_t*)ws.pair_prow, c.T, c.d_model, c.top_k, (const T*)ln.x_raw, ln.stats, ln.gamma, (const T*)ln.dresidual, (T*)dx, ln.partials))
  if (threads == 128) { if (nv == 1) DB(1, 128); else if (nv == 2) DB(2, 128); else return FOMOE_ERR_UNSUPPORTED; }
  else { if (nv == 2) DB(2, 256); else if (nv == 4) DB(4, 256); else return FOMOE_ERR_UNSUPPORTED; }
#undef DB
  FOMOE_LAUNCH_OK("dx_sum_periln_kernel");
  return FOMOE_OK;
}

int launch_dx_sum_periln(const fomoe_config& c, const RouteWs& ws, const void* dxp, const void* dx_sh, const float* dx_r, const void* dx_r_t,
                         const fomoe_periln_pre_bwd& ln, void* dx, cudaStream_t st) {
  const int nb = periln_blocks(c.T);
  if (c.T > 0) {
    int rc = c.dtype == FOMOE_BF16 ? dx_sum_periln_t<__nv_bfloat16>(c, ws, dxp, dx_sh, dx_r, dx_r_t, ln, dx, nb, st)
                                   : dx_sum_periln_t<float>(c, ws, dxp, dx_sh, dx_r, dx_r_t, ln, dx, nb, st);
    if (rc != FOMOE_OK) return rc;
  }
  periln_reduce_kernel<<<ceil_div(c.d_model, 32), 1024, 0, st>>>(ln.partials, c.T > 0 ? nb : 0, c.d_model, ln.dgamma, ln.dbeta);
  FOMOE_LAUNCH_OK("periln_reduce_kernel");
  return FOMOE_OK;
}

}  // namespace fomoe

// ---------------------------------------------------------------------------------------------------------
// Allocation-free Peri-LN backward: fomoe_periln_bwd with its `partials` workspace in a static device array.
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it) and
// so cannot provide fomoe_periln_workspace_bytes() bytes of scratch: the per-CTA dgamma / dbeta partial sums live in the
// array below, 16 MiB that every GPU which loads libfomoe.so holds until the process exits.  Same kernels, same grid and
// same fixed-order reduction as fomoe_periln_bwd: the results are bit-identical to it.
//   * limit: 2 * periln_blocks(T) * d_model <= kNoAllocFloats (periln_blocks = min(T, 4 * SMs): on a 148-SM B200 any T up
//     to d_model = 3543; larger rows only for fewer tokens); beyond it FOMOE_ERR_UNSUPPORTED with a text in fomoe_last_cuda_error().
//   * every call on a device shares the array: calls that overlap on the GPU (different streams, or concurrent graphs) RACE.
//     Calls on one stream are ordered and safe.  Nothing in it has to start at zero -- every CTA of the backward kernel
//     overwrites its own 2 * d_model partials before the reduce kernel reads them -- so the previous call's contents are
//     simply overwritten and no clearing pass is needed.
//   * no cudaMalloc / cudaFree / allocating library call: the only set-up is cudaGetSymbolAddress, once per device.
// In HOST code the array's name is a host-side stand-in for the symbol, not a device address: the kernels get the pointer
// cudaGetSymbolAddress returns for the CURRENT device.
// ---------------------------------------------------------------------------------------------------------
constexpr size_t kNoAllocFloats = (size_t)4 << 20;   // 4 Mi floats = 16 MiB
static __device__ __align__(256) float g_periln_noalloc_scratch[kNoAllocFloats];

static float* periln_noalloc_scratch_ptr(cudaError_t* err) {
  static float* addr[fomoe::kMaxDev] = {};   // per device; racing host threads write the same value
  const int dev = fomoe::current_device();
  *err = cudaSuccess;
  if (!addr[dev]) {
    float* ptr = nullptr;
    *err = cudaGetSymbolAddress((void**)&ptr, g_periln_noalloc_scratch);   // resolves the symbol on the current device
    if (*err != cudaSuccess) return nullptr;
    addr[dev] = ptr;
  }
  return addr[dev];
}

extern "C" FOMOE_API size_t fomoe_periln_bwd_noalloc_max_floats(void) { return kNoAllocFloats; }

extern "C" FOMOE_API int fomoe_periln_bwd_noalloc(int32_t T, int32_t d_model, int32_t dtype, const void* dout, const void* x, const float* stats,
                                                  const float* gamma, float alpha, const void* dresidual, void* dx, float* dgamma,
                                                  float* dbeta, void* stream) {
  using namespace fomoe;
  reset_launch_count();
  if (T < 0 || d_model <= 0 || (dtype != FOMOE_F32 && dtype != FOMOE_BF16) || !gamma || !dgamma || !dbeta) return FOMOE_ERR_BADARG;
  if (T > 0 && (!dout || !x || !stats || !dx)) return FOMOE_ERR_BADARG;
  if (((uintptr_t)dout | (uintptr_t)x | (uintptr_t)dresidual | (uintptr_t)dx | (uintptr_t)gamma) & 15) return FOMOE_ERR_BADARG;
  if ((size_t)d_model * 16 > 200 * 1024) return FOMOE_ERR_UNSUPPORTED;
  const size_t need = 2 * (size_t)periln_blocks(T) * (size_t)d_model;
  if (need > kNoAllocFloats) {
    char msg[256];
    snprintf(msg, sizeof(msg), "fomoe_periln_bwd_noalloc: T = %d, d_model = %d needs %zu floats of scratch, the static array holds %zu "
             "(use fomoe_periln_bwd with a caller-owned workspace)", (int)T, (int)d_model, need, kNoAllocFloats);
    return set_error_text(FOMOE_ERR_UNSUPPORTED, msg);
  }
  cudaError_t e;
  float* partials = periln_noalloc_scratch_ptr(&e);
  if (!partials) return set_cuda_error(e, "cudaGetSymbolAddress(g_periln_noalloc_scratch)");
  note_api_entry("@fomoe_periln_bwd_noalloc", (cudaStream_t)stream);
  return launch_periln_bwd(T, d_model, dtype, dout, x, stats, gamma, alpha, dresidual, dx, dgamma, dbeta, partials, (cudaStream_t)stream);
}
