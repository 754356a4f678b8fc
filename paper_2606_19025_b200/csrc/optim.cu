// Optimizer steps on either side of the resident-delta pack: fused local AdamW over the resident
// experts (Table 7: weight decay 0, betas (0.9, 0.95), eps 1e-8) and the outer Nesterov step
// that consumes the replica-group average of the packed deltas (Alg. 2 l.19-20; server lr 0.7, momentum 0.9).
// Both are pure streaming kernels: 16-byte accesses, one pass, fp32 arithmetic; bound by HBM bandwidth.
#include "common.cuh"

namespace fomoe {
namespace {

constexpr int kOptThreads = 256;

struct AdamArgs {
  float* w[3];
  const void* g[3];
  float* m[3];
  float* v[3];
  void* wc[3];     // compute-dtype copy of w (or nullptr)
  long n[3];       // elements per tensor (all resident slots)
  float lr, beta1, beta2, eps, wd, inv_bc1, inv_bc2;
};

__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, const float4& v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ void st4_bf16(__nv_bfloat16* p, const float4& v) {
  __nv_bfloat162 lo = __floats2bfloat162_rn(v.x, v.y), hi = __floats2bfloat162_rn(v.z, v.w);
  uint2 o;
  o.x = *reinterpret_cast<uint32_t*>(&lo);
  o.y = *reinterpret_cast<uint32_t*>(&hi);
  *reinterpret_cast<uint2*>(p) = o;
}
__device__ __forceinline__ float4 ld4_as_f32(const void* base, long i, bool bf16g) {
  if (!bf16g) return ld4(reinterpret_cast<const float*>(base) + i);
  const uint2 r = *reinterpret_cast<const uint2*>(reinterpret_cast<const __nv_bfloat16*>(base) + i);
  const float2 a = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&r.x));
  const float2 b = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&r.y));
  return make_float4(a.x, a.y, b.x, b.y);
}

// blockIdx.y = tensor (gate, up, down); 4 elements per thread per iteration
template <bool BF16>
__global__ void __launch_bounds__(kOptThreads) adamw_kernel(const AdamArgs a) {
  const int ti = blockIdx.y;
  const long n = a.n[ti];
  float* __restrict__ w = a.w[ti];
  float* __restrict__ m = a.m[ti];
  float* __restrict__ v = a.v[ti];
  const void* __restrict__ g = a.g[ti];
  for (long i = 4 * ((long)blockIdx.x * kOptThreads + threadIdx.x); i < n; i += 4L * gridDim.x * kOptThreads) {
    float4 gw = ld4_as_f32(g, i, BF16), mw = ld4(m + i), vw = ld4(v + i), ww = ld4(w + i);
    float* gp = &gw.x; float* mp = &mw.x; float* vp = &vw.x; float* wp = &ww.x;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      mp[q] = a.beta1 * mp[q] + (1.0f - a.beta1) * gp[q];
      vp[q] = a.beta2 * vp[q] + (1.0f - a.beta2) * gp[q] * gp[q];
      wp[q] -= a.lr * a.wd * wp[q];                                                        // decoupled weight decay
      wp[q] -= a.lr * (mp[q] * a.inv_bc1) / (sqrtf(vp[q] * a.inv_bc2) + a.eps);
    }
    st4(m + i, mw);
    st4(v + i, vw);
    st4(w + i, ww);
    if (a.wc[ti]) {
      if (BF16) st4_bf16(reinterpret_cast<__nv_bfloat16*>(a.wc[ti]) + i, ww);
      else st4(reinterpret_cast<float*>(a.wc[ti]) + i, ww);
    }
  }
}

struct OuterArgs {
  float* w_start[3];
  float* w_now[3];
  float* buf[3];
  void* wc[3];
  long elems[3], off[3], block;   // per-slot elements, offset of the tensor inside a payload block, block size
  float lr, mu;
};

// grid (x, n_pack, 3): packed slot b = blockIdx.y updates resident slot s = pack_slots[b] from payload block b
template <bool BF16>
__global__ void __launch_bounds__(kOptThreads)
outer_nesterov_kernel(const OuterArgs a, const float* __restrict__ payload, const int32_t* __restrict__ pack_slots) {
  const int ti = blockIdx.z, b = blockIdx.y;
  const int s = pack_slots ? pack_slots[b] : b;
  const long n = a.elems[ti];
  const float* __restrict__ dl = payload + (size_t)b * a.block + a.off[ti];
  float* __restrict__ ws = a.w_start[ti] + (size_t)s * n;
  float* __restrict__ wn = a.w_now[ti] + (size_t)s * n;
  float* __restrict__ bu = a.buf[ti] + (size_t)s * n;
  for (long i = 4 * ((long)blockIdx.x * kOptThreads + threadIdx.x); i < n; i += 4L * gridDim.x * kOptThreads) {
    float4 d = ld4(dl + i), mo = ld4(bu + i), w = ld4(ws + i);
    float* dp = &d.x; float* mp = &mo.x; float* wp = &w.x;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      mp[q] = a.mu * mp[q] + dp[q];                      // buf <- mu buf + delta
      wp[q] -= a.lr * (dp[q] + a.mu * mp[q]);            // Nesterov: step along delta + mu buf
    }
    st4(bu + i, mo);
    st4(ws + i, w);
    st4(wn + i, w);
    if (a.wc[ti]) {
      if (BF16) st4_bf16(reinterpret_cast<__nv_bfloat16*>(a.wc[ti]) + (size_t)s * n + i, w);
      else st4(reinterpret_cast<float*>(a.wc[ti]) + (size_t)s * n + i, w);
    }
  }
}

}  // namespace

int launch_adamw(float* const w[3], const void* const g[3], float* const m[3], float* const v[3], void* const wc[3], int dtype,
                 int n_res, const int64_t elems[3], int step, float lr, float b1, float b2, float eps, float wd, cudaStream_t st) {
  AdamArgs a{};
  long nmax = 0;
  for (int i = 0; i < 3; ++i) {
    a.w[i] = w[i]; a.g[i] = g[i]; a.m[i] = m[i]; a.v[i] = v[i]; a.wc[i] = wc ? wc[i] : nullptr;
    a.n[i] = (long)n_res * elems[i];
    if (a.n[i] > nmax) nmax = a.n[i];
  }
  if (nmax == 0) return FOMOE_OK;
  a.lr = lr; a.beta1 = b1; a.beta2 = b2; a.eps = eps; a.wd = wd;
  a.inv_bc1 = (float)(1.0 / (1.0 - pow((double)b1, (double)step)));
  a.inv_bc2 = (float)(1.0 / (1.0 - pow((double)b2, (double)step)));
  long gx = (nmax / 4 + kOptThreads - 1) / kOptThreads;
  if (gx > (long)num_sms() * 8) gx = (long)num_sms() * 8;
  dim3 grid((unsigned)gx, 3);
  if (dtype == FOMOE_BF16) adamw_kernel<true><<<grid, kOptThreads, 0, st>>>(a);
  else adamw_kernel<false><<<grid, kOptThreads, 0, st>>>(a);
  FOMOE_LAUNCH_OK("adamw_kernel");
  return FOMOE_OK;
}

int launch_outer_nesterov(float* const w_start[3], float* const w_now[3], float* const buf[3], void* const wc[3], int dtype,
                          const float* payload, const int64_t elems[3], const int32_t* pack_slots, int n_pack, float lr, float mu,
                          cudaStream_t st) {
  if (n_pack == 0) return FOMOE_OK;
  OuterArgs a{};
  long off = 0, nmax = 0;
  for (int i = 0; i < 3; ++i) {
    a.w_start[i] = w_start[i]; a.w_now[i] = w_now[i]; a.buf[i] = buf[i]; a.wc[i] = wc ? wc[i] : nullptr;
    a.elems[i] = elems[i]; a.off[i] = off;
    off += elems[i];
    if (elems[i] > nmax) nmax = elems[i];
  }
  a.block = off; a.lr = lr; a.mu = mu;
  if (nmax == 0) return FOMOE_OK;
  long gx = (nmax / 4 + kOptThreads - 1) / kOptThreads, want = ((long)num_sms() * 16 + 3L * n_pack - 1) / (3L * n_pack);
  if (gx > want) gx = want;
  if (gx < 1) gx = 1;
  dim3 grid((unsigned)gx, (unsigned)n_pack, 3);
  if (dtype == FOMOE_BF16) outer_nesterov_kernel<true><<<grid, kOptThreads, 0, st>>>(a, payload, pack_slots);
  else outer_nesterov_kernel<false><<<grid, kOptThreads, 0, st>>>(a, payload, pack_slots);
  FOMOE_LAUNCH_OK("outer_nesterov_kernel");
  return FOMOE_OK;
}

}  // namespace fomoe
