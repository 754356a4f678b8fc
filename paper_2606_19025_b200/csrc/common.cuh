// Shared host/device helpers of libfomoe (sm_100a only).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <functional>

#include "../../include/fomoe.h"

namespace fomoe {

constexpr int kTileM = 128;      // rows of one expert-GEMM tile; every slot's row group is padded to this
constexpr int kPermTokens = 128; // tokens (x top_k pairs) handled by one block of the permutation kernels = one router tile
constexpr int kMaxE = 512;
constexpr int kMaxK = 32;

// ---- per-thread error / launch bookkeeping (api.cu) ----
void note_launch(const char* name, cudaStream_t st);   // counts the launch; records a profiling event when enabled
void note_api_entry(const char* name, cudaStream_t st);  // profiling marker at the start of an entry point
int set_cuda_error(cudaError_t e, const char* where);
int set_error_text(int code, const char* text);   // returns `code`; the text is what fomoe_last_cuda_error() then reports
void reset_launch_count();
#define FOMOE_CUDA_OK(expr)                                          \
  do {                                                               \
    cudaError_t e__ = (expr);                                        \
    if (e__ != cudaSuccess) return fomoe::set_cuda_error(e__, #expr); \
  } while (0)
#define FOMOE_LAUNCH_OK(name)                                        \
  do {                                                               \
    fomoe::note_launch(name, st);                                    \
    cudaError_t e__ = cudaGetLastError();                            \
    if (e__ != cudaSuccess) return fomoe::set_cuda_error(e__, name);  \
  } while (0)

// ---- programmatic dependent launch (PDL) ----
// Every kernel of the bf16 path is launched with cudaLaunchAttributeProgrammaticStreamSerialization: its CTAs may become
// resident (and run their prologue: barrier init, TMEM allocation, descriptor prefetch) while the previous kernel on the
// stream is still draining.  The contract that keeps this safe: such a kernel calls pdl_launch_dependents() at its top
// and pdl_wait() BEFORE its first access to global memory; pdl_wait() returns once every earlier grid has completed and
// its writes are visible (so dependencies are transitive along the stream).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
bool pdl_enabled();
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl_enabled() ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// ---- per-device facts (a process may drive several GPUs; host threads may race: the values written are idempotent) ----
constexpr int kMaxDev = 64;
inline int current_device() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDev) dev = 0;
  return dev;
}
inline int num_sms() {   // SM count of the CURRENT device
  static int n[kMaxDev] = {};
  const int dev = current_device();
  if (n[dev] == 0) {
    int v = 148;
    cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
    n[dev] = v;
  }
  return n[dev];
}
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per device: one flag per (kernel instantiation, device)
struct PerDeviceOnce {
  bool done[kMaxDev] = {};
  bool need() const { return !done[current_device()]; }
  void set() { done[current_device()] = true; }
};

inline __host__ __device__ int ceil_div(int a, int b) { return (a + b - 1) / b; }
inline __host__ __device__ size_t align_up(size_t a, size_t b) { return (a + b - 1) / b * b; }

// ---- element access: storage type -> fp32 and back ----
template <typename T> __device__ __forceinline__ float to_f32(T v);
template <> __device__ __forceinline__ float to_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ float to_f32<__nv_bfloat16>(__nv_bfloat16 v) { return __bfloat162float(v); }
template <typename T> __device__ __forceinline__ T from_f32(float v);
template <> __device__ __forceinline__ float from_f32<float>(float v) { return v; }
template <> __device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

__device__ __forceinline__ float sigmoidf_(float v) { return 1.0f / (1.0f + __expf(-v)); }

// ---- layout of fomoe_route_state.internal (all int32 unless noted), computed identically on every call ----
struct RouteWs {
  int32_t* slot_of;     // [E]            resident slot of expert e or -1 (ghost)
  int32_t* blk_hist;    // [n_blk, n_res] kept pairs per (permutation block, slot); then exclusive over blocks
  int32_t* pad_offsets; // [n_res+1]      first padded row of slot s (multiples of kTileM)
  int32_t* pad_end64;   // [n_res]        pad_offsets[s] + count[s] rounded up to 64: end of the K range of the slot's wgrad
  int32_t* n_mtiles;    // [4]            [0] = number of kTileM-row tiles in use, [1] = padded rows in use, [2] = tile pairs
  int32_t* tile_slot;   // [max_mtiles]   slot of row tile i
  int32_t* pair_info;   // [max_mtiles]   CTA-pair work items: 2 * first row tile + (second tile belongs to the same slot)
  int32_t* prow_token;  // [R_cap]        token of padded row r, -1 for padding rows
  float* prow_gate;     // [R_cap]        gate of padded row r
  int32_t* prow_pair;   // [R_cap]        t*k+j of padded row r
  int32_t* pair_prow;   // [T*k]          padded row of pair, -1 if skipped
  void* wr_split;       // [d, 256] bf16  W_r split into bf16 pieces for the tensor-core router
  void* wr_bf;          // [d, Ez] bf16   W_r rounded to bf16, Ez = E rounded up to 64 (tensor-core router backward)
  int n_blk, max_mtiles, R_cap;
  size_t bytes;
};

inline RouteWs carve_route_ws(const fomoe_config& c, int n_res, void* base) {
  RouteWs w{};
  long pairs = (long)c.T * c.top_k;
  w.n_blk = (c.T + kPermTokens - 1) / kPermTokens;
  if (w.n_blk < 1) w.n_blk = 1;
  w.max_mtiles = (int)((pairs + kTileM - 1) / kTileM) + n_res;
  if (w.max_mtiles < 1) w.max_mtiles = 1;
  w.R_cap = w.max_mtiles * kTileM;
  char* p = (char*)base;
  size_t off = 0;
  auto take = [&](size_t n) { void* r = p ? p + off : nullptr; off = align_up(off + n, 256); return r; };
  w.slot_of = (int32_t*)take(sizeof(int32_t) * (size_t)c.E);
  w.blk_hist = (int32_t*)take(sizeof(int32_t) * (size_t)w.n_blk * (size_t)(n_res > 0 ? n_res : 1));
  w.pad_offsets = (int32_t*)take(sizeof(int32_t) * (size_t)(n_res + 1));
  w.pad_end64 = (int32_t*)take(sizeof(int32_t) * (size_t)(n_res > 0 ? n_res : 1));
  w.n_mtiles = (int32_t*)take(sizeof(int32_t) * 4);
  w.tile_slot = (int32_t*)take(sizeof(int32_t) * (size_t)w.max_mtiles);
  w.pair_info = (int32_t*)take(sizeof(int32_t) * (size_t)w.max_mtiles);
  w.prow_token = (int32_t*)take(sizeof(int32_t) * (size_t)w.R_cap);
  w.prow_gate = (float*)take(sizeof(float) * (size_t)w.R_cap);
  w.prow_pair = (int32_t*)take(sizeof(int32_t) * (size_t)w.R_cap);
  w.pair_prow = (int32_t*)take(sizeof(int32_t) * (size_t)(pairs > 0 ? pairs : 1));
  w.wr_split = take(sizeof(__nv_bfloat16) * (size_t)c.d_model * 256);
  w.wr_bf = take(sizeof(__nv_bfloat16) * (size_t)c.d_model * (size_t)((c.E + 63) / 64 * 64));
  w.bytes = off;
  return w;
}

// ---- saved activations (fwd -> bwd) and scratch ----
struct ActWs {
  void* xp;   // [R_cap, d]   gathered token rows (zero for padding rows)
  void* a;    // [R_cap, F]   W_gate x          (tcgen05 path: silu'(a) * u, what the backward multiplies dh with for da)
  void* u;    // [R_cap, F]   W_up x            (tcgen05 path: silu(a), the factor for du)
  void* h;    // [R_cap, F]   silu(a) * u
  void* o;    // [R_cap, d]   W_down h
  void* sa;   // [T, n_sh*F_sh] shared experts: a
  void* su;   // [T, n_sh*F_sh]
  void* sh;   // [T, n_sh*F_sh]
  size_t bytes;
};
inline ActWs carve_act_ws(const fomoe_config& c, int R_cap, void* base) {
  ActWs w{};
  size_t es = c.dtype == FOMOE_BF16 ? 2 : 4;
  char* p = (char*)base;
  size_t off = 0;
  auto take = [&](size_t n) { void* r = p ? p + off : nullptr; off = align_up(off + n, 256); return r; };
  w.xp = take(es * (size_t)R_cap * c.d_model);
  w.a = take(es * (size_t)R_cap * c.d_ff);
  w.u = take(es * (size_t)R_cap * c.d_ff);
  w.h = take(es * (size_t)R_cap * c.d_ff);
  w.o = take(es * (size_t)R_cap * c.d_model);
  size_t fs = (size_t)c.n_shared * c.d_ff_shared;
  w.sa = take(es * (size_t)c.T * fs);
  w.su = take(es * (size_t)c.T * fs);
  w.sh = take(es * (size_t)c.T * fs);
  w.bytes = off;
  return w;
}

struct ScratchWs {
  // forward
  void* y_sh;      // [T, d]  shared-expert output (element type)
  // backward
  void* dop;       // [R_cap, d]  g * dy per padded row
  void* da;        // [R_cap, F]
  void* du;        // [R_cap, F]
  void* dxp;       // [R_cap, d]
  float* dgate;    // [T*k] fp32
  float* dgate_part; // [R_cap, n_dgate_parts] fp32: per padded row, partial <dh, h> sums written by the DH epilogue (two-matrix
                   // expert on the tensor-core path: dgate = sum(parts) / gate, without reading o or dy again)
  int n_dgate_parts; // 2 * ceil(F / 256): two epilogue warps share the 32-column chunks of every 256-column tile
  float* dz;       // [T, E] fp32
  float* dx_r;     // [T, d] fp32  router term dz W_r^T
  void* dsa;       // [T, n_sh*F_sh]
  void* dsu;       // [T, n_sh*F_sh]
  void* dx_sh;     // [T, d]
  float* dwr_part; // [kRouterSplit, d, Ez] fp32 split-K partials of dW_r
  float* wg_tail;  // [SMs / 2 tail tiles * 2 CTAs, 128, 256] fp32 K pieces of the tail tiles of the shared-expert weight gradients (umma_gemm.cu)
  void* dz_bf;     // [T, Ez] bf16 dz, Ez = E rounded up to 64 (tensor-core router backward)
  void* wr_bf;     // [d, Ez] bf16 W_r
  int Ez;
  size_t bytes;
};
constexpr int kRouterSplit = 32;
constexpr int kTailSplitMax = 4;
inline ScratchWs carve_scratch_ws(const fomoe_config& c, int R_cap, void* base) {
  ScratchWs w{};
  size_t es = c.dtype == FOMOE_BF16 ? 2 : 4;
  char* p = (char*)base;
  size_t off = 0;
  auto take = [&](size_t n) { void* r = p ? p + off : nullptr; off = align_up(off + n, 256); return r; };
  size_t fs = (size_t)c.n_shared * c.d_ff_shared;
  w.y_sh = take(es * (size_t)c.T * c.d_model);
  w.dop = take(es * (size_t)R_cap * c.d_model);
  w.da = take(es * (size_t)R_cap * c.d_ff);
  w.du = take(es * (size_t)R_cap * c.d_ff);
  w.dxp = take(es * (size_t)R_cap * c.d_model);
  w.dgate = (float*)take(sizeof(float) * (size_t)c.T * c.top_k);
  w.n_dgate_parts = 2 * ((c.d_ff + 255) / 256);
  w.dgate_part = (float*)take(sizeof(float) * (size_t)R_cap * (size_t)w.n_dgate_parts);
  w.dz = (float*)take(sizeof(float) * (size_t)c.T * c.E);
  w.dx_r = (float*)take(sizeof(float) * (size_t)c.T * c.d_model);
  w.dsa = take(es * (size_t)c.T * fs);
  w.dsu = take(es * (size_t)c.T * fs);
  w.dx_sh = take(es * (size_t)c.T * c.d_model);
  w.Ez = (c.E + 63) / 64 * 64;
  w.dwr_part = (float*)take(sizeof(float) * (size_t)kRouterSplit * c.d_model * w.Ez);
  w.wg_tail = (float*)take(c.n_shared > 0 ? sizeof(float) * (size_t)(num_sms() / 2 + 1) * 2 * 128 * 256 : 0);   // < SMs / 2 tail tiles, each cut into pieces that together fill the pairs
  w.dz_bf = take(sizeof(__nv_bfloat16) * (size_t)c.T * w.Ez);
  w.wr_bf = take(sizeof(__nv_bfloat16) * (size_t)c.d_model * w.Ez);
  w.bytes = off;
  return w;
}

// ---- launchers implemented in the other translation units (all enqueue on `st`, return FOMOE_* status) ----
int launch_route(const fomoe_config& c, const void* x, const float* w_router, const float* bias,
                 const int32_t* resident_ids, int n_res, const fomoe_route_state& out, const RouteWs& ws, cudaStream_t st);
// tensor-core router (route_umma.cu + ROUTE mode of umma_gemm.cu): bf16 tokens, d % 64 == 0, E <= 128, k <= 32
bool route_umma_supported(const fomoe_config& c);
int launch_route_umma(const fomoe_config& c, const void* x, const float* w_router, const float* bias, const int32_t* resident_ids,
                      int n_res, const fomoe_route_state& out, const RouteWs& ws, cudaStream_t st);
bool force_simt();

// row-wise (bandwidth) kernels, rows.cu
int launch_gather_rows(const fomoe_config& c, const void* x, const RouteWs& ws, void* xp, cudaStream_t st);
int launch_combine(const fomoe_config& c, const fomoe_route_state& r, const RouteWs& ws, const void* o, const void* y_sh,
                   void* y, cudaStream_t st);
int launch_combine_bwd(const fomoe_config& c, const void* dy, const void* o, const RouteWs& ws, void* dop, float* dgate,
                       cudaStream_t st);
int launch_scale_rows(const fomoe_config& c, const void* dy, const RouteWs& ws, void* dop, cudaStream_t st);
// dgate_part != nullptr: dgate of a kept pair = sum of its row's n_parts partials / its gate (see ScratchWs::dgate_part);
// n_parts < 0: -n_parts partials that are NOT scaled by the gate (the gathered DH of fine_gemm.cu), no division
int launch_gate_bwd(const fomoe_config& c, const fomoe_route_state& r, const RouteWs& ws, const float* dgate, const float* dgate_part,
                    int n_parts, float* dz, void* dz_bf, int ldz_bf, cudaStream_t st);
int launch_dx_sum(const fomoe_config& c, const RouteWs& ws, const void* dxp, const void* dx_sh, const float* dx_r, const void* dx_r_t,
                  void* dx, cudaStream_t st);

// fp32-accumulate SIMT GEMM path, simt_gemm.cu (all shapes, both dtypes)
struct FfnPtrs {
  const void *w_gate, *w_up, *w_down, *sh_gate, *sh_up, *sh_down;
};
int simt_ffn_fwd(const fomoe_config& c, int n_res, const void* x, const RouteWs& rws, const ActWs& aws, const ScratchWs& sws,
                 const FfnPtrs& w, cudaStream_t st);
int simt_ffn_bwd(const fomoe_config& c, int n_res, const void* x, const void* dy, const RouteWs& rws, const ActWs& aws,
                 const ScratchWs& sws, const FfnPtrs& w, void* dw_gate, void* dw_up, void* dw_down, void* d_sh_gate,
                 void* d_sh_up, void* d_sh_down, cudaStream_t st);
int simt_router_bwd(const fomoe_config& c, const void* x, const float* w_router, const ScratchWs& sws, float* dw_router,
                    cudaStream_t st);

// tcgen05 / TMA grouped GEMM path, umma_gemm.cu (bf16, d % 64 == 0, F % 64 == 0)
bool umma_supported(const fomoe_config& c);
int umma_ffn_fwd(const fomoe_config& c, int n_res, const void* x, const RouteWs& rws, const ActWs& aws, const ScratchWs& sws,
                 const FfnPtrs& w, cudaStream_t st);
// dgate_in_dh: the DH epilogue also writes sws.dgate_part (two-matrix expert only); after_dh, if set, is called right after
// the routed DH launch (the router's backward chain can start there)
int umma_ffn_bwd(const fomoe_config& c, int n_res, const void* x, const void* dy, const RouteWs& rws, const ActWs& aws,
                 const ScratchWs& sws, const FfnPtrs& w, void* dw_gate, void* dw_up, void* dw_down, void* d_sh_gate,
                 void* d_sh_up, void* d_sh_down, cudaStream_t st, bool dgate_in_dh = false,
                 const std::function<int()>* after_dh = nullptr, cudaStream_t wg_stream = nullptr, cudaEvent_t wg_fork = nullptr,
                 bool* wg_forked = nullptr);   // wg_stream: the weight gradients go there, forked (wg_fork) after the last DX launch

// Fine-grained two-matrix experts (d_expert = 128), fine_gemm.cu: the expert GEMMs gather their token-indexed
// operand rows inside the kernel (no permuted copy of x or dy).  fine_mask: which of them apply to this configuration
// (bit 0 = forward GEMM 1, bit 1 = DH, bit 2 = the weight gradients; 0 = none: the grouped kernels of umma_gemm.cu run).
int fine_mask(const fomoe_config& c);
int fine_fwd1(const fomoe_config& c, int n_res, const void* x, const RouteWs& rws, const ActWs& aws, const void* w_up, cudaStream_t st);
int fine_dh(const fomoe_config& c, int n_res, const void* dy, const RouteWs& rws, const ActWs& aws, const ScratchWs& sws, void* hg,
            const void* w_down, cudaStream_t st);
int fine_wgrad(const fomoe_config& c, int n_res, const void* x, const void* dy, const RouteWs& rws, const ScratchWs& sws, const void* hg,
               void* dw_up, void* dw_down, cudaStream_t st);

// F1-F4 on tensor cores (ROUTE mode of the grouped kernel); called by launch_route_umma after the preparation kernel
int umma_route(const fomoe_config& c, const void* x, const void* wr_split, int NP, int Epad, int pieces, const float* bias, int n_res,
               const fomoe_route_state& out, const RouteWs& ws, cudaStream_t st);

// B7 on tensor cores: dx_r (bf16, into sws.dx_r reinterpreted) = dz W_r^T and dW_r = x^T dz (split-K, fp32 partials)
// wr_bf: W_r already rounded to bf16 [d, Ez] by the tensor-core router's preparation kernel, or nullptr (converted here)
int umma_router_bwd(const fomoe_config& c, const void* x, const float* w_router, const void* wr_bf, const ScratchWs& sws,
                    float* dw_router, cudaStream_t st);

// diagnostics (diag.cu)
int launch_routing_stats(const fomoe_config& c, const fomoe_route_state& r, int n_res, int32_t* load, float* stats, cudaStream_t st);
int validate_resident(const int32_t* resident_ids, int n_res, int E, cudaStream_t st, char* msg, size_t msg_len);

int launch_pack(const float* const w_now[3], const float* const w_start[3], int n_res, int64_t eg, int64_t eu, int64_t ed,
                const int32_t* pack_slots, int n_pack, float* payload, cudaStream_t st);

// Peri-LN either side of the block (periln.cu)
int periln_blocks(int T);
int launch_periln_fwd(int T, int d, int dtype, const void* x, const float* gamma, const float* beta, float eps, const void* residual,
                      float alpha, void* out, float* stats, cudaStream_t st);
int launch_periln_bwd(int T, int d, int dtype, const void* dout, const void* x, const float* stats, const float* gamma, float alpha,
                      const void* dresidual, void* dx, float* dgamma, float* dbeta, float* partials, cudaStream_t st);

// fused forms (periln.cu): combine + post-LN + residual, dx scatter-sum + pre-LN backward + residual
bool periln_fused_supported(const fomoe_config& c);
int launch_combine_periln(const fomoe_config& c, const fomoe_route_state& r, const RouteWs& ws, const void* o, const void* y_sh, void* y,
                          const fomoe_periln_post& ln, cudaStream_t st);
int launch_dx_sum_periln(const fomoe_config& c, const RouteWs& ws, const void* dxp, const void* dx_sh, const float* dx_r, const void* dx_r_t,
                         const fomoe_periln_pre_bwd& ln, void* dx, cudaStream_t st);

// optimizer steps around the pack (optim.cu)
int launch_adamw(float* const w[3], const void* const g[3], float* const m[3], float* const v[3], void* const wc[3], int dtype,
                 int n_res, const int64_t elems[3], int step, float lr, float b1, float b2, float eps, float wd, cudaStream_t st);
int launch_outer_nesterov(float* const w_start[3], float* const w_now[3], float* const buf[3], void* const wc[3], int dtype,
                          const float* payload, const int64_t elems[3], const int32_t* pack_slots, int n_pack, float lr, float mu,
                          cudaStream_t st);

}  // namespace fomoe
