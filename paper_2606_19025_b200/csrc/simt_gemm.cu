// fp32-accumulate SIMT grouped GEMMs for the expert FFN, forward and backward (rows F6, F6s, F7, B2-B4, B7 of
// SURVEY.md §8(a)).  This is the fp32 implementation (BASELINE.json config 1 needs true fp32 multiply-add: one tf32
// rounding already costs ~1e-3) and the any-shape path for bf16; the tensor-core path is umma_gemm.cu.
// One 64x64 output tile per 256-thread block, 4x4 outputs per thread, K staged 16 at a time in shared memory.
#include "common.cuh"

namespace fomoe {

constexpr int kBM = 64, kBN = 64, kBK = 16, kPad = 4, kGemmThreads = 256;

struct TileSmem {
  float As[kBK][kBM + kPad];
  float Bs[kBK][kBN + kPad];
};

// acc += A[m0.., 0..K) * B[n0.., 0..K)^T.  A(m,k) = A[m*a_sm + k*a_sk] for m < m_valid (else 0); B likewise.
template <typename TA, typename TB>
__device__ __forceinline__ void tile_acc(float (&acc)[4][4], const TA* __restrict__ A, long a_sm, long a_sk, int m_valid,
                                         const TB* __restrict__ B, long b_sn, long b_sk, int n_valid, int K, TileSmem& sm) {
  const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
  const bool a_kc = (a_sk == 1), b_kc = (b_sk == 1);
  for (int k0 = 0; k0 < K; k0 += kBK) {
#pragma unroll
    for (int i = 0; i < (kBM * kBK) / kGemmThreads; ++i) {
      int idx = tid + i * kGemmThreads;
      int m = a_kc ? idx / kBK : idx % kBM, k = a_kc ? idx % kBK : idx / kBM;
      float v = 0.f;
      if (m < m_valid && k0 + k < K) v = to_f32(A[(long)m * a_sm + (long)(k0 + k) * a_sk]);
      sm.As[k][m] = v;
    }
#pragma unroll
    for (int i = 0; i < (kBN * kBK) / kGemmThreads; ++i) {
      int idx = tid + i * kGemmThreads;
      int n = b_kc ? idx / kBK : idx % kBN, k = b_kc ? idx % kBK : idx / kBN;
      float v = 0.f;
      if (n < n_valid && k0 + k < K) v = to_f32(B[(long)n * b_sn + (long)(k0 + k) * b_sk]);
      sm.Bs[k][n] = v;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < kBK; ++kk) {
      float4 a4 = *reinterpret_cast<const float4*>(&sm.As[kk][ty * 4]);
      float4 b4 = *reinterpret_cast<const float4*>(&sm.Bs[kk][tx * 4]);
      const float a[4] = {a4.x, a4.y, a4.z, a4.w}, b[4] = {b4.x, b4.y, b4.z, b4.w};
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
}

__device__ __forceinline__ void zero_acc(float (&acc)[4][4]) {
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
}

// Row space of a launch: either the tile-padded routed rows (slot per 128-row tile, row count on the device) or
// `dense_rows` dense rows where blockIdx.z selects the shared expert ("part").
struct RowSpace {
  const int32_t* n_mtiles;   // device, [1] = rows in use; NULL for dense
  const int32_t* tile_slot;  // device; NULL for dense
  int dense_rows;
};
__device__ __forceinline__ bool row_tile(const RowSpace& rs, int& row0, int& m_valid, int& slot, int& part) {
  row0 = blockIdx.x * kBM;
  if (rs.tile_slot) {
    if (row0 >= rs.n_mtiles[1]) return false;
    m_valid = kBM;
    slot = rs.tile_slot[row0 / kTileM];
    part = 0;
  } else {
    if (row0 >= rs.dense_rows) return false;
    m_valid = min(kBM, rs.dense_rows - row0);
    slot = blockIdx.z;
    part = blockIdx.z;
  }
  return true;
}

// F6 / F6s: a = X W_g^T, u = X W_u^T, h = silu(a) * u.   X [rows, d]; W [slots, F, d]; outputs [rows, ld] at col part*F.
// Wg == nullptr: the paper's two-matrix expert, a = X W_u^T, h = silu(a); u is not written.
template <typename T>
__global__ void __launch_bounds__(kGemmThreads)
simt_ffn1_kernel(RowSpace rs, const T* __restrict__ X, int d, int F, const T* __restrict__ Wg, const T* __restrict__ Wu, int ld,
                 T* __restrict__ a_out, T* __restrict__ u_out, T* __restrict__ h_out) {
  __shared__ TileSmem sm;
  int row0, m_valid, slot, part;
  if (!row_tile(rs, row0, m_valid, slot, part)) return;
  const int n0 = blockIdx.y * kBN, n_valid = min(kBN, F - n0);
  float ag[4][4], au[4][4];
  zero_acc(ag);
  zero_acc(au);
  const T* A = X + (size_t)row0 * d;
  const bool silu_only = Wg == nullptr;
  tile_acc(ag, A, d, 1, m_valid, (silu_only ? Wu : Wg) + ((size_t)slot * F + n0) * d, d, 1, n_valid, d, sm);
  if (!silu_only) tile_acc(au, A, d, 1, m_valid, Wu + ((size_t)slot * F + n0) * d, d, 1, n_valid, d, sm);
  const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int m = ty * 4 + i, n = tx * 4 + j;
      if (m < m_valid && n < n_valid) {
        size_t off = (size_t)(row0 + m) * ld + (size_t)part * F + n0 + n;
        float av = ag[i][j], uv = silu_only ? 1.0f : au[i][j];
        a_out[off] = from_f32<T>(av);
        if (!silu_only) u_out[off] = from_f32<T>(uv);
        h_out[off] = from_f32<T>(av / (1.0f + expf(-av)) * uv);
      }
    }
}

// F7 / F6s: o[r, :] = sum_parts H[r, part*F : +F] W_d[slot]^T.   W_d [slots, d, F]; out [rows, d].
template <typename T>
__global__ void __launch_bounds__(kGemmThreads)
simt_ffn2_kernel(RowSpace rs, const T* __restrict__ H, int ld, int d, int F, int parts, const T* __restrict__ Wd,
                 T* __restrict__ out) {
  __shared__ TileSmem sm;
  int row0, m_valid, slot, part;
  if (!row_tile(rs, row0, m_valid, slot, part)) return;
  const int n0 = blockIdx.y * kBN, n_valid = min(kBN, d - n0);
  float acc[4][4];
  zero_acc(acc);
  for (int p = 0; p < parts; ++p) {
    int s = rs.tile_slot ? slot : p;
    tile_acc(acc, H + (size_t)row0 * ld + (size_t)p * F, ld, 1, m_valid, Wd + ((size_t)s * d + n0) * F, F, 1, n_valid, F, sm);
  }
  const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int m = ty * 4 + i, n = tx * 4 + j;
      if (m < m_valid && n < n_valid) out[(size_t)(row0 + m) * d + n0 + n] = from_f32<T>(acc[i][j]);
    }
}

// B2 dgrad + B3: dh = dO W_d;  da = dh u s (1 + a (1 - s)), du = dh a s, s = sigmoid(a).
template <typename T>
__global__ void __launch_bounds__(kGemmThreads)
simt_dh_kernel(RowSpace rs, const T* __restrict__ dO, int d, int F, const T* __restrict__ Wd, int ld, const T* __restrict__ a_in,
               const T* __restrict__ u_in, T* __restrict__ da_out, T* __restrict__ du_out) {
  __shared__ TileSmem sm;
  int row0, m_valid, slot, part;
  if (!row_tile(rs, row0, m_valid, slot, part)) return;
  const int n0 = blockIdx.y * kBN, n_valid = min(kBN, F - n0);
  float acc[4][4];
  zero_acc(acc);
  // B(n = f, k = i) = W_d[slot][i][f]
  tile_acc(acc, dO + (size_t)row0 * d, d, 1, m_valid, Wd + (size_t)slot * d * F + n0, 1, F, n_valid, d, sm);
  const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int m = ty * 4 + i, n = tx * 4 + j;
      if (m < m_valid && n < n_valid) {
        size_t off = (size_t)(row0 + m) * ld + (size_t)part * F + n0 + n;
        float av = to_f32(a_in[off]), uv = u_in ? to_f32(u_in[off]) : 1.0f, dh = acc[i][j];   // u_in == nullptr: h = silu(a)
        float s = 1.0f / (1.0f + expf(-av));
        da_out[off] = from_f32<T>(dh * uv * s * (1.0f + av * (1.0f - s)));
        if (u_in) du_out[off] = from_f32<T>(dh * av * s);
      }
    }
}

// B4 dgrad: dxp[r, :] = sum_parts (dA[r, part] W_g[slot] + dU[r, part] W_u[slot]).
template <typename T>
__global__ void __launch_bounds__(kGemmThreads)
simt_dx_kernel(RowSpace rs, const T* __restrict__ dA, const T* __restrict__ dU, int ld, int d, int F, int parts,
               const T* __restrict__ Wg, const T* __restrict__ Wu, T* __restrict__ out) {
  __shared__ TileSmem sm;
  int row0, m_valid, slot, part;
  if (!row_tile(rs, row0, m_valid, slot, part)) return;
  const int n0 = blockIdx.y * kBN, n_valid = min(kBN, d - n0);
  float acc[4][4];
  zero_acc(acc);
  for (int p = 0; p < parts; ++p) {
    int s = rs.tile_slot ? slot : p;
    // B(n = i, k = f) = W[s][f][i]
    if (Wg) {
      tile_acc(acc, dA + (size_t)row0 * ld + (size_t)p * F, ld, 1, m_valid, Wg + (size_t)s * F * d + n0, 1, d, n_valid, F, sm);
      tile_acc(acc, dU + (size_t)row0 * ld + (size_t)p * F, ld, 1, m_valid, Wu + (size_t)s * F * d + n0, 1, d, n_valid, F, sm);
    } else {  // two-matrix expert: dxp = dA W_up
      tile_acc(acc, dA + (size_t)row0 * ld + (size_t)p * F, ld, 1, m_valid, Wu + (size_t)s * F * d + n0, 1, d, n_valid, F, sm);
    }
  }
  const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int m = ty * 4 + i, n = tx * 4 + j;
      if (m < m_valid && n < n_valid) out[(size_t)(row0 + m) * d + n0 + n] = from_f32<T>(acc[i][j]);
    }
}

// wgrad: dW[z][m][n] = sum_{r in rows(z)} A[r, z*a_col + m] * B[r, z*b_col + n].
// rows(z) = [pad_offsets[z], pad_offsets[z+1]) (routed; padding rows are zero), or, with pad_offsets == NULL,
// [z*chunk, min((z+1)*chunk, dense_rows)) if chunk > 0 (split-K partials), else all of [0, dense_rows) (shared experts).
template <typename TA, typename TB, typename TO>
__global__ void __launch_bounds__(kGemmThreads)
simt_wgrad_kernel(const int32_t* __restrict__ pad_offsets, int dense_rows, int chunk, const TA* __restrict__ A, int lda, int a_col,
                  const TB* __restrict__ B, int ldb, int b_col, int M, int N, TO* __restrict__ dW) {
  __shared__ TileSmem sm;
  const int z = blockIdx.z;
  int r0, r1;
  if (pad_offsets) { r0 = pad_offsets[z]; r1 = pad_offsets[z + 1]; }
  else if (chunk > 0) { r0 = min(z * chunk, dense_rows); r1 = min(r0 + chunk, dense_rows); }
  else { r0 = 0; r1 = dense_rows; }
  const int m0 = blockIdx.x * kBM, n0 = blockIdx.y * kBN;
  const int m_valid = min(kBM, M - m0), n_valid = min(kBN, N - n0);
  float acc[4][4];
  zero_acc(acc);
  tile_acc(acc, A + (size_t)r0 * lda + (size_t)z * a_col + m0, 1, lda, m_valid, B + (size_t)r0 * ldb + (size_t)z * b_col + n0, 1, ldb,
           n_valid, r1 - r0, sm);
  const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int m = ty * 4 + i, n = tx * 4 + j;
      if (m < m_valid && n < n_valid) dW[((size_t)z * M + m0 + m) * N + n0 + n] = from_f32<TO>(acc[i][j]);
    }
}

// plain C[M,N] (fp32) = A[M,K] B[N,K]^T, both K-contiguous fp32 (router term dx_r = dz W_r^T).
__global__ void __launch_bounds__(kGemmThreads)
simt_nt_f32_kernel(const float* __restrict__ A, const float* __restrict__ B, int M, int N, int K, float* __restrict__ C) {
  __shared__ TileSmem sm;
  const int m0 = blockIdx.x * kBM, n0 = blockIdx.y * kBN;
  const int m_valid = min(kBM, M - m0), n_valid = min(kBN, N - n0);
  float acc[4][4];
  zero_acc(acc);
  tile_acc(acc, A + (size_t)m0 * K, K, 1, m_valid, B + (size_t)n0 * K, K, 1, n_valid, K, sm);
  const int ty = threadIdx.x >> 4, tx = threadIdx.x & 15;
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int m = ty * 4 + i, n = tx * 4 + j;
      if (m < m_valid && n < n_valid) C[(size_t)(m0 + m) * N + n0 + n] = acc[i][j];
    }
}

// fixed-order reduction of the split-K partials of dW_r
__global__ void reduce_parts_kernel(const float* __restrict__ part, int n_parts, long n, float* __restrict__ out) {
  long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float s = 0.f;
  for (int p = 0; p < n_parts; ++p) s += part[(size_t)p * n + i];
  out[i] = s;
}

// ---------------------------------------------------------------------------------------------------------
template <typename T>
static int ffn_fwd_t(const fomoe_config& c, int n_res, const T* x, const RouteWs& rws, const ActWs& aws, const ScratchWs& sws,
                     const FfnPtrs& w_in, cudaStream_t st) {
  const int d = c.d_model, F = c.d_ff;
  FfnPtrs w = w_in;
  if (c.expert_fn == FOMOE_EXPERT_SILU) w.w_gate = w.sh_gate = nullptr;   // whatever was passed is ignored (fomoe.h)
  if (n_res > 0 && c.T > 0) {
    RowSpace rs{rws.n_mtiles, rws.tile_slot, 0};
    dim3 g1(rws.R_cap / kBM, ceil_div(F, kBN));
    simt_ffn1_kernel<T><<<g1, kGemmThreads, 0, st>>>(rs, (const T*)aws.xp, d, F, (const T*)w.w_gate, (const T*)w.w_up, F, (T*)aws.a,
                                                     (T*)aws.u, (T*)aws.h);
    FOMOE_LAUNCH_OK("simt_ffn1_kernel");
    dim3 g2(rws.R_cap / kBM, ceil_div(d, kBN));
    simt_ffn2_kernel<T><<<g2, kGemmThreads, 0, st>>>(rs, (const T*)aws.h, F, d, F, 1, (const T*)w.w_down, (T*)aws.o);
    FOMOE_LAUNCH_OK("simt_ffn2_kernel");
  }
  if (c.n_shared > 0 && c.T > 0) {
    const int Fs = c.d_ff_shared, ld = c.n_shared * Fs;
    RowSpace rs{nullptr, nullptr, c.T};
    dim3 g1(ceil_div(c.T, kBM), ceil_div(Fs, kBN), c.n_shared);
    simt_ffn1_kernel<T><<<g1, kGemmThreads, 0, st>>>(rs, x, d, Fs, (const T*)w.sh_gate, (const T*)w.sh_up, ld, (T*)aws.sa, (T*)aws.su,
                                                     (T*)aws.sh);
    FOMOE_LAUNCH_OK("simt_ffn1_kernel(shared)");
    dim3 g2(ceil_div(c.T, kBM), ceil_div(d, kBN), 1);
    simt_ffn2_kernel<T><<<g2, kGemmThreads, 0, st>>>(rs, (const T*)aws.sh, ld, d, Fs, c.n_shared, (const T*)w.sh_down, (T*)sws.y_sh);
    FOMOE_LAUNCH_OK("simt_ffn2_kernel(shared)");
  }
  return FOMOE_OK;
}

int simt_ffn_fwd(const fomoe_config& c, int n_res, const void* x, const RouteWs& rws, const ActWs& aws, const ScratchWs& sws,
                 const FfnPtrs& w, cudaStream_t st) {
  return c.dtype == FOMOE_BF16 ? ffn_fwd_t<__nv_bfloat16>(c, n_res, (const __nv_bfloat16*)x, rws, aws, sws, w, st)
                               : ffn_fwd_t<float>(c, n_res, (const float*)x, rws, aws, sws, w, st);
}

template <typename T>
static int ffn_bwd_t(const fomoe_config& c, int n_res, const T* x, const T* dy, const RouteWs& rws, const ActWs& aws,
                     const ScratchWs& sws, const FfnPtrs& w_in, T* dw_gate, T* dw_up, T* dw_down, T* d_sh_gate, T* d_sh_up,
                     T* d_sh_down, cudaStream_t st) {
  const int d = c.d_model, F = c.d_ff;
  const bool silu = c.expert_fn == FOMOE_EXPERT_SILU;   // two-matrix expert: no gate path, dW_up = dA^T x
  FfnPtrs w = w_in;
  if (silu) w.w_gate = w.sh_gate = nullptr;
  if (n_res > 0) {
    RowSpace rs{rws.n_mtiles, rws.tile_slot, 0};
    if (c.T > 0) {
      dim3 g1(rws.R_cap / kBM, ceil_div(F, kBN));
      simt_dh_kernel<T><<<g1, kGemmThreads, 0, st>>>(rs, (const T*)sws.dop, d, F, (const T*)w.w_down, F, (const T*)aws.a,
                                                     silu ? nullptr : (const T*)aws.u, (T*)sws.da, (T*)sws.du);
      FOMOE_LAUNCH_OK("simt_dh_kernel");
      dim3 g2(rws.R_cap / kBM, ceil_div(d, kBN));
      simt_dx_kernel<T><<<g2, kGemmThreads, 0, st>>>(rs, (const T*)sws.da, (const T*)sws.du, F, d, F, 1, (const T*)w.w_gate,
                                                     (const T*)w.w_up, (T*)sws.dxp);
      FOMOE_LAUNCH_OK("simt_dx_kernel");
    }
    // weight gradients per resident slot (T == 0 or an empty slot gives exact zeros)
    dim3 gd(ceil_div(d, kBM), ceil_div(F, kBN), n_res);
    simt_wgrad_kernel<T, T, T><<<gd, kGemmThreads, 0, st>>>(rws.pad_offsets, 0, 0, (const T*)sws.dop, d, 0, (const T*)aws.h, F, 0, d, F,
                                                            dw_down);
    FOMOE_LAUNCH_OK("simt_wgrad_kernel(down)");
    dim3 gg(ceil_div(F, kBM), ceil_div(d, kBN), n_res);
    if (!silu) {
      simt_wgrad_kernel<T, T, T><<<gg, kGemmThreads, 0, st>>>(rws.pad_offsets, 0, 0, (const T*)sws.da, F, 0, (const T*)aws.xp, d, 0, F, d,
                                                              dw_gate);
      FOMOE_LAUNCH_OK("simt_wgrad_kernel(gate)");
    }
    simt_wgrad_kernel<T, T, T><<<gg, kGemmThreads, 0, st>>>(rws.pad_offsets, 0, 0, (const T*)(silu ? sws.da : sws.du), F, 0, (const T*)aws.xp, d, 0, F, d,
                                                            dw_up);
    FOMOE_LAUNCH_OK("simt_wgrad_kernel(up)");
  }
  if (c.n_shared > 0) {
    const int Fs = c.d_ff_shared, ld = c.n_shared * Fs;
    RowSpace rs{nullptr, nullptr, c.T};
    if (c.T > 0) {
      dim3 g1(ceil_div(c.T, kBM), ceil_div(Fs, kBN), c.n_shared);
      simt_dh_kernel<T><<<g1, kGemmThreads, 0, st>>>(rs, dy, d, Fs, (const T*)w.sh_down, ld, (const T*)aws.sa, silu ? nullptr : (const T*)aws.su,
                                                     (T*)sws.dsa, (T*)sws.dsu);
      FOMOE_LAUNCH_OK("simt_dh_kernel(shared)");
      dim3 g2(ceil_div(c.T, kBM), ceil_div(d, kBN), 1);
      simt_dx_kernel<T><<<g2, kGemmThreads, 0, st>>>(rs, (const T*)sws.dsa, (const T*)sws.dsu, ld, d, Fs, c.n_shared, (const T*)w.sh_gate,
                                                     (const T*)w.sh_up, (T*)sws.dx_sh);
      FOMOE_LAUNCH_OK("simt_dx_kernel(shared)");
    }
    // one z-slice per shared expert, each over all T rows (chunk = 0)
    dim3 gd(ceil_div(d, kBM), ceil_div(Fs, kBN), c.n_shared);
    simt_wgrad_kernel<T, T, T><<<gd, kGemmThreads, 0, st>>>(nullptr, c.T, 0, dy, d, 0, (const T*)aws.sh, ld, Fs, d, Fs, d_sh_down);
    FOMOE_LAUNCH_OK("simt_wgrad_kernel(sh_down)");
    dim3 gg(ceil_div(Fs, kBM), ceil_div(d, kBN), c.n_shared);
    if (!silu) {
      simt_wgrad_kernel<T, T, T><<<gg, kGemmThreads, 0, st>>>(nullptr, c.T, 0, (const T*)sws.dsa, ld, Fs, x, d, 0, Fs, d, d_sh_gate);
      FOMOE_LAUNCH_OK("simt_wgrad_kernel(sh_gate)");
    }
    simt_wgrad_kernel<T, T, T><<<gg, kGemmThreads, 0, st>>>(nullptr, c.T, 0, (const T*)(silu ? sws.dsa : sws.dsu), ld, Fs, x, d, 0, Fs, d, d_sh_up);
    FOMOE_LAUNCH_OK("simt_wgrad_kernel(sh_up)");
  }
  return FOMOE_OK;
}

int simt_ffn_bwd(const fomoe_config& c, int n_res, const void* x, const void* dy, const RouteWs& rws, const ActWs& aws,
                 const ScratchWs& sws, const FfnPtrs& w, void* dw_gate, void* dw_up, void* dw_down, void* d_sh_gate,
                 void* d_sh_up, void* d_sh_down, cudaStream_t st) {
  if (c.dtype == FOMOE_BF16) {
    using T = __nv_bfloat16;
    return ffn_bwd_t<T>(c, n_res, (const T*)x, (const T*)dy, rws, aws, sws, w, (T*)dw_gate, (T*)dw_up, (T*)dw_down, (T*)d_sh_gate,
                        (T*)d_sh_up, (T*)d_sh_down, st);
  }
  using T = float;
  return ffn_bwd_t<T>(c, n_res, (const T*)x, (const T*)dy, rws, aws, sws, w, (T*)dw_gate, (T*)dw_up, (T*)dw_down, (T*)d_sh_gate,
                      (T*)d_sh_up, (T*)d_sh_down, st);
}

// B7: dW_r = x^T dz (split over tokens, fixed-order reduce) and dx_r = dz W_r^T.
int simt_router_bwd(const fomoe_config& c, const void* x, const float* w_router, const ScratchWs& sws, float* dw_router,
                    cudaStream_t st) {
  const int d = c.d_model, E = c.E;
  const int chunk = ceil_div(c.T > 0 ? c.T : 1, kRouterSplit);
  dim3 g(ceil_div(d, kBM), ceil_div(E, kBN), kRouterSplit);
  if (c.dtype == FOMOE_BF16)
    simt_wgrad_kernel<__nv_bfloat16, float, float><<<g, kGemmThreads, 0, st>>>(nullptr, c.T, chunk, (const __nv_bfloat16*)x, d, 0, sws.dz, E,
                                                                             0, d, E, sws.dwr_part);
  else
    simt_wgrad_kernel<float, float, float><<<g, kGemmThreads, 0, st>>>(nullptr, c.T, chunk, (const float*)x, d, 0, sws.dz, E, 0, d, E,
                                                                     sws.dwr_part);
  FOMOE_LAUNCH_OK("simt_wgrad_kernel(router)");
  long n = (long)d * E;
  reduce_parts_kernel<<<(int)((n + 255) / 256), 256, 0, st>>>(sws.dwr_part, kRouterSplit, n, dw_router);
  FOMOE_LAUNCH_OK("reduce_parts_kernel");
  if (c.T > 0) {
    dim3 g2(ceil_div(c.T, kBM), ceil_div(d, kBN));
    simt_nt_f32_kernel<<<g2, kGemmThreads, 0, st>>>(sws.dz, w_router, c.T, d, E, sws.dx_r);
    FOMOE_LAUNCH_OK("simt_nt_f32_kernel");
  }
  return FOMOE_OK;
}

}  // namespace fomoe
