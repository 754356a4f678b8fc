// extern "C" entry points of libfomoe (include/fomoe.h): argument checks, workspace carving, kernel sequencing.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <atomic>
#include <functional>
#include <vector>

#include "common.cuh"

namespace fomoe {

static thread_local char g_err[512] = "";
static thread_local int g_launches = 0;
static std::atomic<int> g_force_simt{0};

// optional per-kernel timing: one event after every launch (+ a marker at each entry point); kernel i's time is the
// interval since the previous event on the same stream
struct ProfRec { const char* name; cudaEvent_t ev; };
static thread_local std::vector<ProfRec> g_prof;
static thread_local bool g_prof_on = false;
static void prof_push(const char* name, cudaStream_t st) {
  cudaEvent_t e;
  if (cudaEventCreate(&e) != cudaSuccess) return;
  cudaEventRecord(e, st);
  g_prof.push_back({name, e});
}
void note_launch(const char* name, cudaStream_t st) {
  ++g_launches;
  if (g_prof_on) prof_push(name, st);
}
void note_api_entry(const char* name, cudaStream_t st) {
  if (g_prof_on) prof_push(name, st);
}
int set_cuda_error(cudaError_t e, const char* where) {
  snprintf(g_err, sizeof(g_err), "%s: %s (%s)", where, cudaGetErrorName(e), cudaGetErrorString(e));
  return FOMOE_ERR_CUDA;
}
// for entry points that live in another translation unit (fomoe_periln_bwd_noalloc, periln.cu)
int set_error_text(int code, const char* text) {
  snprintf(g_err, sizeof(g_err), "%s", text);
  return code;
}
void reset_launch_count() { g_launches = 0; }

// The one piece of state the library owns: a side stream and two events per host thread, used by fomoe_moe_bwd to run the
// router's backward chain (gate_bwd, dz W_r^T, x^T dz) beside the expert GEMMs.  Fork / join through events, so the pattern
// is capturable in a CUDA graph.  FOMOE_SIDE_STREAM=0 in the environment turns it off.
struct SideStream {
  cudaStream_t s = nullptr;
  cudaEvent_t fork = nullptr, join = nullptr;
  // a second one for the weight-gradient GEMMs of the tensor-core path: they depend on DH only, so they run beside the
  // bandwidth-bound dx scatter-sum (which co-resides with their one-CTA-per-SM kernels) instead of ahead of it
  cudaStream_t s2 = nullptr;
  cudaEvent_t fork2 = nullptr, join2 = nullptr;
  bool ok = false;
};
constexpr int kMaxDevices = 64;
static thread_local SideStream g_side[kMaxDevices];   // one per (host thread, device): a device switch creates, never leaks
static bool wg_stream_enabled() {   // FOMOE_WG_STREAM=0: weight gradients on the caller's stream, no stream priorities
  static const bool on = [] { const char* e = getenv("FOMOE_WG_STREAM"); return !(e && e[0] == '0'); }();
  return on;
}
static bool side_enabled() {
  static const bool on = [] { const char* e = getenv("FOMOE_SIDE_STREAM"); return !(e && e[0] == '0'); }();
  return on;
}
static SideStream* side_stream() {
  if (!side_enabled() || g_prof_on) return nullptr;   // per-kernel timing needs one serial stream
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
  SideStream& sd = g_side[dev];
  if (!sd.ok) {
    // priorities: the router's backward chain first (the dx scatter-sum waits for it, and its GEMMs need whole SMs), the
    // weight gradients last (nothing in the step waits for them), so that when the DX kernel drains the chain gets the SMs
    int prio_lo = 0, prio_hi = 0;
    if (wg_stream_enabled()) cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);   // (numerically: lowest priority = largest value)
    if (!sd.s && cudaStreamCreateWithPriority(&sd.s, cudaStreamNonBlocking, prio_hi) != cudaSuccess) return nullptr;
    if (!sd.fork && cudaEventCreateWithFlags(&sd.fork, cudaEventDisableTiming) != cudaSuccess) return nullptr;
    if (!sd.join && cudaEventCreateWithFlags(&sd.join, cudaEventDisableTiming) != cudaSuccess) return nullptr;
    if (!sd.s2 && cudaStreamCreateWithPriority(&sd.s2, cudaStreamNonBlocking, prio_lo) != cudaSuccess) return nullptr;
    if (!sd.fork2 && cudaEventCreateWithFlags(&sd.fork2, cudaEventDisableTiming) != cudaSuccess) return nullptr;
    if (!sd.join2 && cudaEventCreateWithFlags(&sd.join2, cudaEventDisableTiming) != cudaSuccess) return nullptr;
    sd.ok = true;
  }
  return &sd;
}

// State of fomoe_moe_step_host, per (host thread, device): a download stream (device -> host copies run on their own copy
// engine, beside the uploads and the kernels) and one event per staging-buffer ADDRESS seen, which orders a call after the
// previous call's use of the same buffer.  Addresses are only compared, never dereferenced.
struct HostPipe {
  cudaStream_t dl = nullptr;
  cudaEvent_t joined = nullptr;
  struct Slot { const void* p; cudaEvent_t ev; };
  std::vector<Slot> slots;
  cudaEvent_t event_of(const void* p) {
    for (auto& sl : slots)
      if (sl.p == p) return sl.ev;
    if (slots.size() >= 64) {                     // a caller cycling through many buffers: forget the oldest (its event is long done)
      cudaEventDestroy(slots.front().ev);
      slots.erase(slots.begin());
    }
    cudaEvent_t e = nullptr;
    if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return nullptr;
    slots.push_back({p, e});
    return e;
  }
};
static thread_local HostPipe g_pipe[kMaxDevices];
static HostPipe* host_pipe() {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
  HostPipe& hp = g_pipe[dev];
  if (!hp.dl && cudaStreamCreateWithFlags(&hp.dl, cudaStreamNonBlocking) != cudaSuccess) return nullptr;
  if (!hp.joined && cudaEventCreateWithFlags(&hp.joined, cudaEventDisableTiming) != cudaSuccess) return nullptr;
  return &hp;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int check_cfg(const fomoe_config* c, int n_res) {
  if (!c) return FOMOE_ERR_BADARG;
  if (c->T < 0 || c->d_model <= 0 || c->E <= 0 || c->top_k <= 0 || c->d_ff <= 0) return FOMOE_ERR_BADARG;
  if (c->top_k > c->E || n_res < 0 || n_res > c->E) return FOMOE_ERR_BADARG;
  if (c->n_shared < 0 || (c->n_shared > 0 && c->d_ff_shared <= 0)) return FOMOE_ERR_BADARG;
  if (c->dtype != FOMOE_F32 && c->dtype != FOMOE_BF16) return FOMOE_ERR_BADARG;
  if (c->gate_fn != FOMOE_GATE_SOFTMAX && c->gate_fn != FOMOE_GATE_SIGMOID) return FOMOE_ERR_BADARG;
  if (c->gate_rule < FOMOE_DROP_ONLY || c->gate_rule > FOMOE_RENORM_RESIDENT) return FOMOE_ERR_BADARG;
  if (!(c->temperature > 0.f)) return FOMOE_ERR_BADARG;
  if (c->expert_fn != FOMOE_EXPERT_SWIGLU && c->expert_fn != FOMOE_EXPERT_SILU) return FOMOE_ERR_BADARG;
  if (c->route_mode != FOMOE_ROUTE_SKIP_TOKEN && c->route_mode != FOMOE_ROUTE_FORCED_LOCAL) return FOMOE_ERR_BADARG;
  if (c->route_mode == FOMOE_ROUTE_FORCED_LOCAL && c->top_k > n_res) return FOMOE_ERR_BADARG;   // bounded by min(k, N_le)
  if (c->E > kMaxE || c->top_k > kMaxK) return FOMOE_ERR_UNSUPPORTED;
  if ((long)c->T * c->top_k + (long)kTileM * (n_res + 1) > 0x7fffffffL / 2) return FOMOE_ERR_UNSUPPORTED;  // int32 row ids
  return FOMOE_OK;
}

bool force_simt() { return g_force_simt != 0; }
// FOMOE_PDL=0 in the environment turns programmatic dependent launch off (A/B measurements, debugging)
bool pdl_enabled() {
  static const bool on = [] { const char* e = getenv("FOMOE_PDL"); return !(e && e[0] == '0'); }();
  return on;
}
static bool use_umma(const fomoe_config& c) { return !g_force_simt && umma_supported(c); }

}  // namespace fomoe

using namespace fomoe;

extern "C" {

int fomoe_abi_version(void) { return FOMOE_ABI_VERSION; }
const char* fomoe_last_cuda_error(void) { return g_err; }
int fomoe_last_launch_count(void) { return g_launches; }
int fomoe_set_force_simt(int on) { return g_force_simt.exchange(on ? 1 : 0); }

int fomoe_profile_enable(int on) {
  for (auto& r : g_prof) cudaEventDestroy(r.ev);
  g_prof.clear();
  g_prof_on = on != 0;
  return FOMOE_OK;
}

int fomoe_profile_collect(const char** names, float* ms, int cap) {
  int n = 0;
  if (!g_prof.empty()) cudaEventSynchronize(g_prof.back().ev);
  for (size_t i = 1; i < g_prof.size(); ++i) {
    if (g_prof[i].name[0] == '@') continue;  // entry marker: the gap before it is not kernel time
    float t = 0.f;
    if (cudaEventElapsedTime(&t, g_prof[i - 1].ev, g_prof[i].ev) != cudaSuccess) t = -1.f;
    if (n < cap) { names[n] = g_prof[i].name; ms[n] = t; }
    ++n;
  }
  for (auto& r : g_prof) cudaEventDestroy(r.ev);
  g_prof.clear();
  return n;
}

int fomoe_workspace_bytes(const fomoe_config* cfg, int32_t n_res, size_t* route_internal, size_t* saved_acts, size_t* scratch) {
  int rc = check_cfg(cfg, n_res);
  if (rc != FOMOE_OK) return rc;
  RouteWs r = carve_route_ws(*cfg, n_res, nullptr);
  if (route_internal) *route_internal = r.bytes;
  if (saved_acts) *saved_acts = carve_act_ws(*cfg, r.R_cap, nullptr).bytes;
  if (scratch) *scratch = carve_scratch_ws(*cfg, r.R_cap, nullptr).bytes;
  return FOMOE_OK;
}

int fomoe_route(const fomoe_config* cfg, const void* x, const float* w_router, const float* router_bias,
                const int32_t* resident_ids, int32_t n_res, const fomoe_route_state* out, void* stream) {
  g_launches = 0;
  int rc = check_cfg(cfg, n_res);
  if (rc != FOMOE_OK) return rc;
  if (!out || !w_router || (!x && cfg->T > 0) || (n_res > 0 && !resident_ids)) return FOMOE_ERR_BADARG;
  if (!out->offsets || !out->internal || (n_res > 0 && !out->counts)) return FOMOE_ERR_BADARG;
  if (cfg->T > 0 && (!out->topk_idx || !out->gate || !out->probs || !out->row_token || !out->pair_row)) return FOMOE_ERR_BADARG;
  if (!aligned16(x) || !aligned16(w_router) || !aligned16(out->internal)) return FOMOE_ERR_BADARG;
  RouteWs ws = carve_route_ws(*cfg, n_res, out->internal);
  note_api_entry("@fomoe_route", (cudaStream_t)stream);
  return launch_route(*cfg, x, w_router, router_bias, resident_ids, n_res, *out, ws, (cudaStream_t)stream);
}

static int moe_fwd_impl(const fomoe_config* cfg, const void* x, const fomoe_route_state* route, int32_t n_res, const void* w_gate,
                        const void* w_up, const void* w_down, const void* sh_gate, const void* sh_up, const void* sh_down, void* y,
                        void* saved_acts, void* scratch, const fomoe_periln_post* ln, void* stream) {
  g_launches = 0;
  int rc = check_cfg(cfg, n_res);
  if (rc != FOMOE_OK) return rc;
  if (!route || !route->internal || !saved_acts || !scratch || ((!x || !y) && cfg->T > 0)) return FOMOE_ERR_BADARG;
  const bool swiglu = cfg->expert_fn == FOMOE_EXPERT_SWIGLU;   // the paper's two-matrix expert has no W_gate
  if (n_res > 0 && ((swiglu && !w_gate) || !w_up || !w_down)) return FOMOE_ERR_BADARG;
  if (cfg->n_shared > 0 && ((swiglu && !sh_gate) || !sh_up || !sh_down)) return FOMOE_ERR_BADARG;
  if (!aligned16(x) || !aligned16(y) || !aligned16(saved_acts) || !aligned16(scratch) || !aligned16(w_gate) || !aligned16(w_up) ||
      !aligned16(w_down) || !aligned16(sh_gate) || !aligned16(sh_up) || !aligned16(sh_down))
    return FOMOE_ERR_BADARG;
  cudaStream_t st = (cudaStream_t)stream;
  RouteWs rws = carve_route_ws(*cfg, n_res, route->internal);
  ActWs aws = carve_act_ws(*cfg, rws.R_cap, saved_acts);
  ScratchWs sws = carve_scratch_ws(*cfg, rws.R_cap, scratch);
  FfnPtrs w{w_gate, w_up, w_down, sh_gate, sh_up, sh_down};
  note_api_entry("@fomoe_moe_fwd", st);
  if (cfg->T == 0) return FOMOE_OK;
  // the permuted copy of x: not needed when both of its readers (forward GEMM 1, dW_up) gather their rows themselves
  const int fine = use_umma(*cfg) ? fine_mask(*cfg) : 0;
  if (n_res > 0 && (fine & 5) != 5) {
    rc = launch_gather_rows(*cfg, x, rws, aws.xp, st);
    if (rc != FOMOE_OK) return rc;
  }
  rc = use_umma(*cfg) ? umma_ffn_fwd(*cfg, n_res, x, rws, aws, sws, w, st) : simt_ffn_fwd(*cfg, n_res, x, rws, aws, sws, w, st);
  if (rc != FOMOE_OK) return rc;
  if (ln) return launch_combine_periln(*cfg, *route, rws, aws.o, cfg->n_shared > 0 ? sws.y_sh : nullptr, y, *ln, st);
  return launch_combine(*cfg, *route, rws, aws.o, cfg->n_shared > 0 ? sws.y_sh : nullptr, y, st);
}

int fomoe_moe_fwd(const fomoe_config* cfg, const void* x, const fomoe_route_state* route, int32_t n_res, const void* w_gate,
                  const void* w_up, const void* w_down, const void* sh_gate, const void* sh_up, const void* sh_down, void* y,
                  void* saved_acts, void* scratch, void* stream) {
  return moe_fwd_impl(cfg, x, route, n_res, w_gate, w_up, w_down, sh_gate, sh_up, sh_down, y, saved_acts, scratch, nullptr, stream);
}

int fomoe_moe_fwd_periln(const fomoe_config* cfg, const void* x, const fomoe_route_state* route, int32_t n_res, const void* w_gate,
                         const void* w_up, const void* w_down, const void* sh_gate, const void* sh_up, const void* sh_down, void* y,
                         void* saved_acts, void* scratch, const fomoe_periln_post* ln, void* stream) {
  if (!cfg || !ln || !ln->gamma || !ln->beta || !(ln->eps >= 0.f)) return FOMOE_ERR_BADARG;
  if (cfg->T > 0 && (!ln->residual || !ln->out || !ln->stats)) return FOMOE_ERR_BADARG;
  if (!aligned16(ln->residual) || !aligned16(ln->out) || !aligned16(ln->gamma) || !aligned16(ln->beta)) return FOMOE_ERR_BADARG;
  if (cfg->d_model > 0 && (cfg->dtype == FOMOE_F32 || cfg->dtype == FOMOE_BF16) && !periln_fused_supported(*cfg)) return FOMOE_ERR_UNSUPPORTED;
  return moe_fwd_impl(cfg, x, route, n_res, w_gate, w_up, w_down, sh_gate, sh_up, sh_down, y, saved_acts, scratch, ln, stream);
}

static int moe_bwd_impl(const fomoe_config* cfg, const void* dy, const void* x, const fomoe_route_state* route, int32_t n_res,
                        const float* w_router, const void* w_gate, const void* w_up, const void* w_down, const void* sh_gate,
                        const void* sh_up, const void* sh_down, const void* saved_acts, void* dx, float* dw_router, void* dw_gate,
                        void* dw_up, void* dw_down, void* d_sh_gate, void* d_sh_up, void* d_sh_down, void* scratch,
                        const fomoe_periln_pre_bwd* ln, void* stream) {
  g_launches = 0;
  int rc = check_cfg(cfg, n_res);
  if (rc != FOMOE_OK) return rc;
  if (!route || !route->internal || !saved_acts || !scratch || !w_router || !dw_router) return FOMOE_ERR_BADARG;
  if (cfg->T > 0 && (!dy || !x || !dx)) return FOMOE_ERR_BADARG;
  const bool swiglu = cfg->expert_fn == FOMOE_EXPERT_SWIGLU;
  if (n_res > 0 && ((swiglu && (!w_gate || !dw_gate)) || !w_up || !w_down || !dw_up || !dw_down)) return FOMOE_ERR_BADARG;
  if (cfg->n_shared > 0 && ((swiglu && (!sh_gate || !d_sh_gate)) || !sh_up || !sh_down || !d_sh_up || !d_sh_down)) return FOMOE_ERR_BADARG;
  if (!aligned16(dy) || !aligned16(x) || !aligned16(dx) || !aligned16(dw_router) || !aligned16(dw_gate) || !aligned16(dw_up) ||
      !aligned16(dw_down) || !aligned16(d_sh_gate) || !aligned16(d_sh_up) || !aligned16(d_sh_down) || !aligned16(scratch) ||
      !aligned16(saved_acts))
    return FOMOE_ERR_BADARG;
  cudaStream_t st = (cudaStream_t)stream;
  RouteWs rws = carve_route_ws(*cfg, n_res, route->internal);
  ActWs aws = carve_act_ws(*cfg, rws.R_cap, const_cast<void*>(saved_acts));
  ScratchWs sws = carve_scratch_ws(*cfg, rws.R_cap, scratch);
  FfnPtrs w{w_gate, w_up, w_down, sh_gate, sh_up, sh_down};
  note_api_entry("@fomoe_moe_bwd", st);
  // B1: do = g dy per row, dgate = <dy, o>.  Two-matrix expert on the tensor-core path: <dy, o> = <dh, h> / g falls out of the
  // DH epilogue (dh = do W_down is there in fp32 and F is narrow), so B1 neither reads o nor reduces: one pass over [P, d] less
  const bool tc_router = use_umma(*cfg) && cfg->T > 0;
  const bool dgate_in_dh = tc_router && n_res > 0 && cfg->expert_fn == FOMOE_EXPERT_SILU;
  const int fine = tc_router ? fine_mask(*cfg) : 0;   // (fine_gemm.cu: bit 1 = DH gathers dy rows, bit 2 = so do the weight gradients)
  if (n_res > 0 && cfg->T > 0 && (fine & 6) == 6) {
    // no B1 kernel at all: the gate scales DH's accumulator, dgate is DH's <dh, h>
  } else if (n_res > 0 && cfg->T > 0) {
    rc = dgate_in_dh ? launch_scale_rows(*cfg, dy, rws, sws.dop, st) : launch_combine_bwd(*cfg, dy, aws.o, rws, sws.dop, sws.dgate, st);
    if (rc != FOMOE_OK) return rc;
  } else {
    FOMOE_CUDA_OK(cudaMemsetAsync(sws.dgate, 0, sizeof(float) * (size_t)cfg->T * cfg->top_k, st));
  }
  // B6, B7 depend only on dgate: on the tensor-core path they run on the side stream, beside B2-B4 (forked after B1, or after
  // the DH launch when that is where dgate comes from)
  SideStream* side = tc_router ? side_stream() : nullptr;
  cudaStream_t rst = side ? side->s : st;
  auto router_bwd = [&]() -> int {
    int r = launch_gate_bwd(*cfg, *route, rws, sws.dgate, dgate_in_dh ? sws.dgate_part : nullptr,
                            (fine & 2) ? -sws.n_dgate_parts : sws.n_dgate_parts, sws.dz,
                            tc_router ? sws.dz_bf : nullptr, sws.Ez, rst);
    if (r != FOMOE_OK) return r;
    // (the tensor-core router of fomoe_route left W_r in bf16 in the route workspace)
    return tc_router ? umma_router_bwd(*cfg, x, w_router, route_umma_supported(*cfg) ? rws.wr_bf : nullptr, sws, dw_router, rst)
                     : simt_router_bwd(*cfg, x, w_router, sws, dw_router, rst);
  };
  bool forked = false, wg_forked = false;
  const bool wg_overlap = wg_stream_enabled();
  auto fork_router = [&]() -> int {   // side stream: waits for everything queued on `st` so far, then runs the router's backward
    FOMOE_CUDA_OK(cudaEventRecord(side->fork, st));
    FOMOE_CUDA_OK(cudaStreamWaitEvent(side->s, side->fork, 0));
    forked = true;
    return router_bwd();
  };
  const std::function<int()> after_dh = [&]() -> int { return side ? fork_router() : FOMOE_OK; };
  // everything between the fork and the join: whatever it returns, the side stream is joined back into `st` afterwards (an
  // error return must not leave a forked stream dangling, least of all inside a stream capture)
  auto forked_region = [&]() -> int {
    int r = FOMOE_OK;
    if (side && !dgate_in_dh) {
      r = fork_router();
      if (r != FOMOE_OK) return r;
    }
    // B2-B4 (+ shared experts)
    r = use_umma(*cfg) ? umma_ffn_bwd(*cfg, n_res, x, dy, rws, aws, sws, w, dw_gate, dw_up, dw_down, d_sh_gate, d_sh_up, d_sh_down, st,
                                      dgate_in_dh, dgate_in_dh ? &after_dh : nullptr, (side && wg_overlap && cfg->T > 0) ? side->s2 : nullptr,
                                      side ? side->fork2 : nullptr, &wg_forked)
                       : simt_ffn_bwd(*cfg, n_res, x, dy, rws, aws, sws, w, dw_gate, dw_up, dw_down, d_sh_gate, d_sh_up, d_sh_down, st);
    if (r != FOMOE_OK) return r;
    return forked ? FOMOE_OK : router_bwd();
  };
  rc = forked_region();
  if (side && forked) {
    cudaError_t e1 = cudaEventRecord(side->join, side->s);
    cudaError_t e2 = cudaStreamWaitEvent(st, side->join, 0);
    if (rc == FOMOE_OK && e1 != cudaSuccess) return set_cuda_error(e1, "cudaEventRecord(join)");
    if (rc == FOMOE_OK && e2 != cudaSuccess) return set_cuda_error(e2, "cudaStreamWaitEvent(join)");
  }
  // B5 (with the pre-LN backward folded in when asked for); whatever happened, the weight-gradient stream is joined back
  if (rc == FOMOE_OK)
    rc = ln ? launch_dx_sum_periln(*cfg, rws, sws.dxp, cfg->n_shared > 0 ? sws.dx_sh : nullptr, tc_router ? nullptr : sws.dx_r,
                                   tc_router ? (const void*)sws.dx_r : nullptr, *ln, dx, st)
            : launch_dx_sum(*cfg, rws, sws.dxp, cfg->n_shared > 0 ? sws.dx_sh : nullptr, tc_router ? nullptr : sws.dx_r,
                            tc_router ? (const void*)sws.dx_r : nullptr, dx, st);
  if (side && wg_forked) {
    cudaError_t e1 = cudaEventRecord(side->join2, side->s2);
    cudaError_t e2 = cudaStreamWaitEvent(st, side->join2, 0);
    if (rc == FOMOE_OK && e1 != cudaSuccess) return set_cuda_error(e1, "cudaEventRecord(join2)");
    if (rc == FOMOE_OK && e2 != cudaSuccess) return set_cuda_error(e2, "cudaStreamWaitEvent(join2)");
  }
  return rc;
}

int fomoe_moe_bwd(const fomoe_config* cfg, const void* dy, const void* x, const fomoe_route_state* route, int32_t n_res,
                  const float* w_router, const void* w_gate, const void* w_up, const void* w_down, const void* sh_gate,
                  const void* sh_up, const void* sh_down, const void* saved_acts, void* dx, float* dw_router, void* dw_gate,
                  void* dw_up, void* dw_down, void* d_sh_gate, void* d_sh_up, void* d_sh_down, void* scratch, void* stream) {
  return moe_bwd_impl(cfg, dy, x, route, n_res, w_router, w_gate, w_up, w_down, sh_gate, sh_up, sh_down, saved_acts, dx, dw_router, dw_gate,
                      dw_up, dw_down, d_sh_gate, d_sh_up, d_sh_down, scratch, nullptr, stream);
}

int fomoe_moe_bwd_periln(const fomoe_config* cfg, const void* dy, const void* x, const fomoe_route_state* route, int32_t n_res,
                         const float* w_router, const void* w_gate, const void* w_up, const void* w_down, const void* sh_gate,
                         const void* sh_up, const void* sh_down, const void* saved_acts, void* dx, float* dw_router, void* dw_gate,
                         void* dw_up, void* dw_down, void* d_sh_gate, void* d_sh_up, void* d_sh_down, void* scratch,
                         const fomoe_periln_pre_bwd* ln, void* stream) {
  if (!cfg || !ln || !ln->gamma || !ln->dgamma || !ln->dbeta || !ln->partials) return FOMOE_ERR_BADARG;
  if (cfg->T > 0 && (!ln->x_raw || !ln->stats)) return FOMOE_ERR_BADARG;
  if (!aligned16(ln->x_raw) || !aligned16(ln->dresidual) || !aligned16(ln->gamma)) return FOMOE_ERR_BADARG;
  if (cfg->d_model > 0 && (cfg->dtype == FOMOE_F32 || cfg->dtype == FOMOE_BF16) && !periln_fused_supported(*cfg)) return FOMOE_ERR_UNSUPPORTED;
  return moe_bwd_impl(cfg, dy, x, route, n_res, w_router, w_gate, w_up, w_down, sh_gate, sh_up, sh_down, saved_acts, dx, dw_router, dw_gate,
                      dw_up, dw_down, d_sh_gate, d_sh_up, d_sh_down, scratch, ln, stream);
}

int fomoe_pack_resident_deltas(const float* const w_now[3], const float* const w_start[3], int32_t n_res, int64_t elems_gate,
                               int64_t elems_up, int64_t elems_down, const int32_t* pack_slots, int32_t n_pack, float* payload,
                               void* stream) {
  g_launches = 0;
  if (!w_now || !w_start || n_res < 0 || n_pack < 0 || elems_gate < 0 || elems_up < 0 || elems_down < 0) return FOMOE_ERR_BADARG;
  if (!pack_slots && n_pack != n_res) return FOMOE_ERR_BADARG;
  if (n_pack == 0) return FOMOE_OK;
  if (!payload || !aligned16(payload)) return FOMOE_ERR_BADARG;
  const int64_t elems[3] = {elems_gate, elems_up, elems_down};
  for (int i = 0; i < 3; ++i) {   // a tensor of zero elements may be NULL (two-matrix expert: no gate block)
    if (elems[i] > 0 && (!w_now[i] || !w_start[i])) return FOMOE_ERR_BADARG;
    if (!aligned16(w_now[i]) || !aligned16(w_start[i])) return FOMOE_ERR_BADARG;
  }
  if (elems_gate % 4 || elems_up % 4 || elems_down % 4) return FOMOE_ERR_UNSUPPORTED;
  note_api_entry("@fomoe_pack_resident_deltas", (cudaStream_t)stream);
  return launch_pack(w_now, w_start, n_res, elems_gate, elems_up, elems_down, pack_slots, n_pack, payload, (cudaStream_t)stream);
}

int fomoe_debug_validate_resident(const int32_t* resident_ids, int32_t n_res, int32_t E, void* stream) {
  if (n_res < 0 || E <= 0 || n_res > E || (n_res > 0 && !resident_ids)) return FOMOE_ERR_BADARG;
  return validate_resident(resident_ids, n_res, E, (cudaStream_t)stream, g_err, sizeof(g_err));
}

int fomoe_routing_stats(const fomoe_config* cfg, const fomoe_route_state* route, int32_t n_res, int32_t* load, float* stats,
                        void* stream) {
  g_launches = 0;
  int rc = check_cfg(cfg, n_res);
  if (rc != FOMOE_OK) return rc;
  if (!route || !load || !stats || !route->offsets || (cfg->T > 0 && (!route->topk_idx || !route->pair_row))) return FOMOE_ERR_BADARG;
  return launch_routing_stats(*cfg, *route, n_res, load, stats, (cudaStream_t)stream);
}

int fomoe_periln_workspace_bytes(int32_t T, int32_t d_model, size_t* partials) {
  if (T < 0 || d_model <= 0 || !partials) return FOMOE_ERR_BADARG;
  *partials = sizeof(float) * 2 * (size_t)periln_blocks(T) * (size_t)d_model;
  return FOMOE_OK;
}

int fomoe_periln_fwd(int32_t T, int32_t d_model, int32_t dtype, const void* x, const float* gamma, const float* beta, float eps,
                     const void* residual, float alpha, void* out, float* stats, void* stream) {
  g_launches = 0;
  if (T < 0 || d_model <= 0 || (dtype != FOMOE_F32 && dtype != FOMOE_BF16) || !gamma || !beta || !(eps >= 0.f)) return FOMOE_ERR_BADARG;
  if (T > 0 && (!x || !out || !stats)) return FOMOE_ERR_BADARG;
  if (!aligned16(x) || !aligned16(out) || !aligned16(residual) || !aligned16(gamma) || !aligned16(beta)) return FOMOE_ERR_BADARG;
  if ((size_t)d_model * 16 > 200 * 1024) return FOMOE_ERR_UNSUPPORTED;   // the backward stages 4 fp32 rows in shared memory
  note_api_entry("@fomoe_periln_fwd", (cudaStream_t)stream);
  return launch_periln_fwd(T, d_model, dtype, x, gamma, beta, eps, residual, alpha, out, stats, (cudaStream_t)stream);
}

int fomoe_periln_bwd(int32_t T, int32_t d_model, int32_t dtype, const void* dout, const void* x, const float* stats, const float* gamma,
                     float alpha, const void* dresidual, void* dx, float* dgamma, float* dbeta, float* partials, void* stream) {
  g_launches = 0;
  if (T < 0 || d_model <= 0 || (dtype != FOMOE_F32 && dtype != FOMOE_BF16) || !gamma || !dgamma || !dbeta || !partials) return FOMOE_ERR_BADARG;
  if (T > 0 && (!dout || !x || !stats || !dx)) return FOMOE_ERR_BADARG;
  if (!aligned16(dout) || !aligned16(x) || !aligned16(dresidual) || !aligned16(dx) || !aligned16(gamma) || !aligned16(partials)) return FOMOE_ERR_BADARG;
  if ((size_t)d_model * 16 > 200 * 1024) return FOMOE_ERR_UNSUPPORTED;
  note_api_entry("@fomoe_periln_bwd", (cudaStream_t)stream);
  return launch_periln_bwd(T, d_model, dtype, dout, x, stats, gamma, alpha, dresidual, dx, dgamma, dbeta, partials, (cudaStream_t)stream);
}

int fomoe_adamw_resident(float* const w_master[3], const void* const grad[3], float* const m[3], float* const v[3],
                         void* const w_compute[3], int32_t dtype, int32_t n_res, int64_t elems_gate, int64_t elems_up,
                         int64_t elems_down, int32_t step, float lr, float beta1, float beta2, float eps, float weight_decay,
                         void* stream) {
  g_launches = 0;
  if (!w_master || !grad || !m || !v || n_res < 0 || step < 1 || elems_gate < 0 || elems_up < 0 || elems_down < 0) return FOMOE_ERR_BADARG;
  if (dtype != FOMOE_F32 && dtype != FOMOE_BF16) return FOMOE_ERR_BADARG;
  if (!(beta1 >= 0.f && beta1 < 1.f && beta2 >= 0.f && beta2 < 1.f) || !(eps >= 0.f)) return FOMOE_ERR_BADARG;
  const int64_t elems[3] = {elems_gate, elems_up, elems_down};
  for (int i = 0; i < 3; ++i) {
    if (elems[i] % 4) return FOMOE_ERR_UNSUPPORTED;
    if (elems[i] > 0 && n_res > 0 && (!w_master[i] || !grad[i] || !m[i] || !v[i])) return FOMOE_ERR_BADARG;
    if (!aligned16(w_master[i]) || !aligned16(grad[i]) || !aligned16(m[i]) || !aligned16(v[i]) || (w_compute && !aligned16(w_compute[i])))
      return FOMOE_ERR_BADARG;
  }
  note_api_entry("@fomoe_adamw_resident", (cudaStream_t)stream);
  return launch_adamw(w_master, grad, m, v, w_compute, dtype, n_res, elems, step, lr, beta1, beta2, eps, weight_decay, (cudaStream_t)stream);
}

int fomoe_outer_nesterov(float* const w_start[3], float* const w_now[3], float* const momentum[3], void* const w_compute[3],
                         int32_t dtype, const float* payload_avg, int32_t n_res, int64_t elems_gate, int64_t elems_up,
                         int64_t elems_down, const int32_t* pack_slots, int32_t n_pack, float lr, float mu, void* stream) {
  g_launches = 0;
  if (!w_start || !w_now || !momentum || n_res < 0 || n_pack < 0 || elems_gate < 0 || elems_up < 0 || elems_down < 0) return FOMOE_ERR_BADARG;
  if (dtype != FOMOE_F32 && dtype != FOMOE_BF16) return FOMOE_ERR_BADARG;
  if (!pack_slots && n_pack != n_res) return FOMOE_ERR_BADARG;
  if (n_pack == 0) return FOMOE_OK;
  if (!payload_avg || !aligned16(payload_avg)) return FOMOE_ERR_BADARG;
  const int64_t elems[3] = {elems_gate, elems_up, elems_down};
  for (int i = 0; i < 3; ++i) {
    if (elems[i] % 4) return FOMOE_ERR_UNSUPPORTED;
    if (elems[i] > 0 && (!w_start[i] || !w_now[i] || !momentum[i])) return FOMOE_ERR_BADARG;
    if (!aligned16(w_start[i]) || !aligned16(w_now[i]) || !aligned16(momentum[i]) || (w_compute && !aligned16(w_compute[i])))
      return FOMOE_ERR_BADARG;
  }
  note_api_entry("@fomoe_outer_nesterov", (cudaStream_t)stream);
  return launch_outer_nesterov(w_start, w_now, momentum, w_compute, dtype, payload_avg, elems, pack_slots, n_pack, lr, mu,
                               (cudaStream_t)stream);
}

int fomoe_moe_step_host(const fomoe_config* cfg, const void* x_host, const void* dy_host, void* y_host, void* dx_host, void* x_dev,
                        void* dy_dev, void* y_dev, void* dx_dev, const float* w_router, const float* router_bias,
                        const int32_t* resident_ids, int32_t n_res, const fomoe_route_state* route, const void* w_gate,
                        const void* w_up, const void* w_down, const void* sh_gate, const void* sh_up, const void* sh_down,
                        float* dw_router, void* dw_gate, void* dw_up, void* dw_down, void* d_sh_gate, void* d_sh_up, void* d_sh_down,
                        void* saved_acts, void* scratch, void* stream, void* copy_stream, int32_t defer_join) {
  int rc = check_cfg(cfg, n_res);
  if (rc != FOMOE_OK) return rc;
  if (!x_host || !dy_host || !y_host || !dx_host || !x_dev || !dy_dev || !y_dev || !dx_dev) return FOMOE_ERR_BADARG;
  cudaStream_t st = (cudaStream_t)stream, cs = (cudaStream_t)copy_stream;
  const size_t bytes = (size_t)cfg->T * cfg->d_model * (cfg->dtype == FOMOE_BF16 ? 2 : 4);
  HostPipe* hp = host_pipe();
  if (!hp) return set_cuda_error(cudaErrorUnknown, "fomoe_moe_step_host: download stream");
  cudaStream_t dl = hp->dl;
  // last use of each staging buffer by an earlier call of this thread: uploads wait for the readers of x_dev / dy_dev, the
  // kernels that overwrite y_dev / dx_dev wait for their previous download.  (Never-recorded events are no-ops to wait on.)
  cudaEvent_t e_x = hp->event_of(x_dev), e_dy = hp->event_of(dy_dev), e_y = hp->event_of(y_dev), e_dx = hp->event_of(dx_dev);
  if (!e_x || !e_dy || !e_y || !e_dx) return set_cuda_error(cudaErrorUnknown, "fomoe_moe_step_host: events");
  int launches = 0;
  struct Events {   // destroyed on every exit path (destroying a pending event is deferred by the runtime)
    cudaEvent_t xup = nullptr, dyup = nullptr, y = nullptr, dx = nullptr;
    ~Events() {
      for (cudaEvent_t e : {xup, dyup, y, dx})
        if (e) cudaEventDestroy(e);
    }
  } ev;
  FOMOE_CUDA_OK(cudaEventCreateWithFlags(&ev.xup, cudaEventDisableTiming));
  FOMOE_CUDA_OK(cudaEventCreateWithFlags(&ev.dyup, cudaEventDisableTiming));
  FOMOE_CUDA_OK(cudaEventCreateWithFlags(&ev.y, cudaEventDisableTiming));
  FOMOE_CUDA_OK(cudaEventCreateWithFlags(&ev.dx, cudaEventDisableTiming));
  // uploads (copy stream): x, then dy -- the second one overlaps route + forward; with alternating staging buffers both
  // overlap the PREVIOUS call's compute
  FOMOE_CUDA_OK(cudaStreamWaitEvent(cs, e_x, 0));
  FOMOE_CUDA_OK(cudaMemcpyAsync(x_dev, x_host, bytes, cudaMemcpyHostToDevice, cs));
  FOMOE_CUDA_OK(cudaEventRecord(ev.xup, cs));
  FOMOE_CUDA_OK(cudaStreamWaitEvent(cs, e_dy, 0));
  FOMOE_CUDA_OK(cudaMemcpyAsync(dy_dev, dy_host, bytes, cudaMemcpyHostToDevice, cs));
  FOMOE_CUDA_OK(cudaEventRecord(ev.dyup, cs));
  auto body = [&]() -> int {
    FOMOE_CUDA_OK(cudaStreamWaitEvent(st, ev.xup, 0));
    FOMOE_CUDA_OK(cudaStreamWaitEvent(st, e_y, 0));
    int r = fomoe_route(cfg, x_dev, w_router, router_bias, resident_ids, n_res, route, st);
    launches += g_launches;
    if (r != FOMOE_OK) return r;
    r = fomoe_moe_fwd(cfg, x_dev, route, n_res, w_gate, w_up, w_down, sh_gate, sh_up, sh_down, y_dev, saved_acts, scratch, st);
    launches += g_launches;
    if (r != FOMOE_OK) return r;
    FOMOE_CUDA_OK(cudaEventRecord(ev.y, st));
    FOMOE_CUDA_OK(cudaStreamWaitEvent(dl, ev.y, 0));
    FOMOE_CUDA_OK(cudaMemcpyAsync(y_host, y_dev, bytes, cudaMemcpyDeviceToHost, dl));  // overlaps the backward
    FOMOE_CUDA_OK(cudaEventRecord(e_y, dl));
    FOMOE_CUDA_OK(cudaStreamWaitEvent(st, ev.dyup, 0));
    FOMOE_CUDA_OK(cudaStreamWaitEvent(st, e_dx, 0));
    r = fomoe_moe_bwd(cfg, dy_dev, x_dev, route, n_res, w_router, w_gate, w_up, w_down, sh_gate, sh_up, sh_down, saved_acts, dx_dev,
                      dw_router, dw_gate, dw_up, dw_down, d_sh_gate, d_sh_up, d_sh_down, scratch, st);
    launches += g_launches;
    if (r != FOMOE_OK) return r;
    FOMOE_CUDA_OK(cudaEventRecord(e_x, st));    // x_dev and dy_dev have been read for the last time
    FOMOE_CUDA_OK(cudaEventRecord(e_dy, st));
    FOMOE_CUDA_OK(cudaEventRecord(ev.dx, st));
    FOMOE_CUDA_OK(cudaStreamWaitEvent(dl, ev.dx, 0));
    FOMOE_CUDA_OK(cudaMemcpyAsync(dx_host, dx_dev, bytes, cudaMemcpyDeviceToHost, dl));  // overlaps the NEXT call's compute
    FOMOE_CUDA_OK(cudaEventRecord(e_dx, dl));
    return FOMOE_OK;
  };
  rc = body();
  // whatever happened, `st` is ordered after the uploads it may not have waited for yet (no dangling work on the copy stream)
  cudaError_t e0 = cudaStreamWaitEvent(st, ev.dyup, 0);
  if (rc == FOMOE_OK && e0 != cudaSuccess) rc = set_cuda_error(e0, "cudaStreamWaitEvent(copy join)");
  if (!defer_join) {
    int jr = fomoe_moe_step_host_join(stream);
    if (rc == FOMOE_OK) rc = jr;
  }
  g_launches = launches;
  return rc;
}

int fomoe_moe_step_host_join(void* stream) {
  HostPipe* hp = host_pipe();
  if (!hp) return set_cuda_error(cudaErrorUnknown, "fomoe_moe_step_host_join: download stream");
  FOMOE_CUDA_OK(cudaEventRecord(hp->joined, hp->dl));
  FOMOE_CUDA_OK(cudaStreamWaitEvent((cudaStream_t)stream, hp->joined, 0));
  return FOMOE_OK;
}

}  // extern "C"
