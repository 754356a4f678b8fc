// tcgen05 / TMEM / TMA grouped GEMMs for the resident-expert SwiGLU FFN, forward and backward
// (rows F6, F6s, F7, B2, B3, B4 of SURVEY.md §8(a)); bf16 operands, fp32 accumulation in tensor memory.
//
// One persistent, warp-specialised kernel template.  CTAs run as PAIRS (cluster of 2 on one TPC, cta_group::2): one
// tcgen05.mma covers 256 rows x 256 columns, each CTA staging its own 128 rows of A and HALF of the columns of B, so
// shared-memory and L2 operand traffic per flop is 2/3 of the single-CTA 128 x 256 tile.  Per CTA, 256 threads:
//   warp 0  : TMA producer   (cp.async.bulk.tensor.2d -> 128B-swizzled shared-memory stages; both CTAs' loads signal
//                             the LEADER's mbarrier with complete_tx)
//   warp 1  : MMA issuer     (leader CTA only: one elected lane issues tcgen05.mma.cta_group::2.kind::f16, M=256 N<=256
//                             K=16; tcgen05.commit multicasts stage release / accumulator-full to both CTAs)
//   warp 2  : TMEM allocator (512 columns = two 128x256 fp32 accumulator stages per CTA)
//   warps 4-7: epilogue      (tcgen05.ld 32x32b -> registers -> fused math -> 16-byte global stores of this CTA's rows)
// Three pipelines: shared-memory full/empty (TMA <-> MMA), TMEM full/empty (MMA <-> epilogue), static round-robin
// tile scheduler over clusters.  The number of row tiles is data dependent and is read from device memory (route
// workspace): the host never learns P.
//
// Modes (pair tile 256 x 256, K staged 64 at a time):
//   FWD1  [a|u] = X W_gate^T | X W_up^T   (A, B K-major; CTA0 stages W_gate, CTA1 W_up; epilogue: h = silu(a)*u, and
//                                           for the backward silu'(a)*u and silu(a) in place of a and u)
//   FWD2  o = H W_down^T                  (A, B K-major)
//   FWD1S a = X W_up^T                    (the paper's two-matrix expert: epilogue h = silu(a), and silu'(a) for
//                                           the backward; loads like FWD2 with K = d)
//   DH    dh = dO W_down                  (A K-major, B MN-major; epilogue: da = dh * silu'(a)u, du = dh * silu(a))
//   DX    dxp = dA W_gate + dU W_up       (A K-major, B MN-major; two K segments into one accumulator)
//   WGRAD dW[g] = A[rows(g)]^T B[rows(g)] (A, B MN-major; K = the group's (padded) rows)
// Row space is either the tile-padded routed rows (pairs of 128-row tiles of ONE slot; the last pair of a slot may hold a
// single tile, then CTA 1 computes rows nobody stores) or dense rows (shared experts).
#include <cuda.h>
#include <stdlib.h>

#include "common.cuh"
#include "umma_ptx.cuh"

namespace fomoe {
namespace {

constexpr int BM = 128;   // rows per CTA (256 per pair)
constexpr int BN = 256;   // accumulator columns (each CTA stages BN/2 columns of B)
constexpr int BK = 64, kAccStages = 2;
constexpr int kABytes = BM * BK * 2, kBBytes = (BN / 2) * BK * 2, kStageBytes = kABytes + kBBytes;
constexpr int kThreads = 384;   // warps 0-3: TMA, MMA, TMEM allocator, idle; warps 4-11: epilogue
constexpr int kEpiWarps = 8;    // two warps per TMEM lane quarter; they take alternate 32-column chunks of a tile
// epilogue staging: per epilogue warp, swizzled tiles of 32 rows x 32 bf16 (2 KB each) used to turn the
// row-per-thread TMEM layout into coalesced 16-byte global accesses
constexpr int kStgTile = 2048;
constexpr int kDhDepth = 3;  // DH epilogue: chunks of (a, u) kept in flight per warp with cp.async
enum Mode { FWD1 = 0, FWD2 = 1, DH = 2, DX = 3, WGRAD = 4, ROUTE = 5, FWD1S = 6 };
// ROUTE epilogue scratch (struct RouteSmem<KMAX> below): slot map, per-stage histograms, top-k candidate / merge lists.  Its size
// follows the list capacity, so that the short lists (k <= 8: 30 KB) leave room for a sixth TMA stage.
__host__ __device__ constexpr int route_stg_bytes(int kmax) {
  const int kn = kmax > 16 ? 16 : (kmax < 2 ? 2 : kmax);
  const int net = kn * 128 * 8 + (kn + 1) * 256 * 8, ins = kmax > 16 ? 2 * kmax * 128 * 4 : 0;
  return (4096 + (net > ins ? net : ins) + 1023) / 1024 * 1024;
}
// DH and FWD1 trade TMA stages for epilogue staging: DH streams a and u back in through a cp.async ring
__host__ __device__ constexpr int stages_of(int mode, int kmax = 0) {
  return mode == DH ? 4 : mode == ROUTE ? (route_stg_bytes(kmax) <= 32768 ? 6 : 5) : (mode == FWD1 || mode == FWD1S) ? 5 : 6;
}
__host__ __device__ constexpr int stg_tiles_per_warp(int mode) { return mode == DH ? 2 * kDhDepth : mode == FWD1 ? 3 : 2; }   // FWD2 / DX: two tiles, alternating under the bulk stores
__host__ __device__ constexpr int stg_bytes_of(int mode, int kmax = 0) {
  return mode == ROUTE ? route_stg_bytes(kmax) : kEpiWarps * stg_tiles_per_warp(mode) * kStgTile;
}
__host__ __device__ constexpr int smem_bytes_of(int mode, int kmax = 0) {
  return stages_of(mode, kmax) * kStageBytes + stg_bytes_of(mode, kmax) + 1024 /*align*/ + 256 /*barriers*/;
}
constexpr int kTmemCols = 512;

struct TmaMaps {
  CUtensorMap m[6];   // WGRAD with several jobs: (A, B) of job j at m[2j], m[2j+1].  FWD2 / DX: m[4] = the output, for the bulk-store epilogue
};

// ROUTE mode (rows F1-F4 + the per-block histogram of F5): everything the router epilogue needs
struct RouteEpi {
  int E, Epad, pieces, k, gate_fn, gate_rule, n_res, forced_local;
  float inv_tau;
  const float* bias;
  const int32_t* slot_of;
  float* probs;
  int32_t* topk_idx;
  float* gate;
  int32_t* blk_hist;  // [ceil(T / 128), n_res]
};

struct UmmaParams {
  const int32_t* n_mtiles;     // routed: device, [2] = tile pairs in use; nullptr = dense rows
  const int32_t* tile_slot;    // routed: slot of row tile
  const int32_t* pair_info;    // routed: 2 * first row tile + (second tile in the same slot)
  const int32_t* pad_offsets;  // routed WGRAD: first padded row of group g
  const int32_t* pad_end64;    // routed WGRAD: end of group g's K range (count rounded up to BK; the rows up to it are zero padding)
  int dense_rows;              // dense: number of rows (T)
  int parts;                   // dense: number of shared experts (1 for routed)
  int n_groups;                // WGRAD: number of groups (n_res or n_shared)
  int d, F;                    // model width; per-expert hidden width
  int ld;                      // leading dimension of the [rows, hidden] activations (F, or parts*F for dense)
  int M, N;                    // WGRAD: output rows / cols per group
  int a_gcol, b_gcol;          // WGRAD dense: per-group column offset into A / B
  int ksegs;                   // DX: K segments (2: dA W_gate + dU W_up; 1: dA W_up, two-matrix expert)
  int k_chunk;                 // WGRAD dense: > 0 = split-K, group g reduces rows [g*k_chunk, (g+1)*k_chunk)
  int tma_store;               // FWD2 / DX: the epilogue stores its 32 x 32 chunks with TMA bulk stores through maps.m[4]
  float* out_f32;              // WGRAD: if set, fp32 output [n_groups, M, N] instead of out0
  // WGRAD dense, tail split: the tiles of the last, partially filled round of the persistent schedule (tile ids >= tail_first)
  // are cut into tail_ks K ranges of tail_chunk rows each, so that round takes 1 / tail_ks of a tile time; the pieces go to
  // tail_part as fp32 [piece][cta][128][256] and wgrad_tail_fixup_kernel adds them in a fixed order
  int tail_first, tail_ks, tail_chunk;
  float* tail_part;
  bf16 *out0, *out1, *out2;    // FWD1: a,u,h | FWD2/DX: out | DH: da,du | WGRAD: dW
  const bf16 *in0, *in1;       // DH: a,u
  const bf16* in_h;            // DH, two-matrix expert (in1 == nullptr): the saved h, streamed in u's ring slot, for
  float* dgate_part;           //   dgate_part[row, 2 n_tile + half] = sum over this warp's chunks of dh * h  (ScratchWs::dgate_part)
  int n_dgate_parts;
  RouteEpi r;                  // ROUTE
  // WGRAD, several weight gradients of the same row groups in ONE launch (dW_down, dW_gate, dW_up): n_jobs > 0 overrides
  // M, N, out0; job j reads tensor maps m[2j] (A) and m[2j+1] (B).  One launch instead of three saves two kernel prologues
  // and tails and lets the jobs fill each other's last scheduler round.
  int n_jobs;
  int job_M[3], job_N[3], job_agcol[3], job_bgcol[3];   // (per-group column offsets into A / B: dense rows, shared experts)
  bf16* job_out[3];
};

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, bool valid) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(valid ? 16 : 0) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- per-warp staging tile: 32 rows x 64 B, two rows per 128-byte line, 16-byte chunks XOR-swizzled so that both the
// row-per-lane accesses and the 8-rows-x-4-chunks global-side accesses are bank-conflict free.  Addresses are
// shared-state-space (ld.shared / st.shared), not generic ----
__device__ __forceinline__ uint32_t stg_off(int r, int q) { return (uint32_t)((r >> 1) * 128 + (((((r & 1) << 2) | q) ^ ((r >> 1) & 7)) * 16)); }
__device__ __forceinline__ void sts128(uint32_t addr, const uint4& v) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&h);
}
__device__ __forceinline__ float2 unpack_bf16x2(uint32_t w) {
  return __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&w));
}

// lane = row: write 32 fp32 as bf16 into the staging tile
__device__ __forceinline__ void stg_put_row(uint32_t stg, int lane, const float (&v)[32]) {
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    uint4 w;
    w.x = pack_bf16x2(v[q * 8 + 0], v[q * 8 + 1]);
    w.y = pack_bf16x2(v[q * 8 + 2], v[q * 8 + 3]);
    w.z = pack_bf16x2(v[q * 8 + 4], v[q * 8 + 5]);
    w.w = pack_bf16x2(v[q * 8 + 6], v[q * 8 + 7]);
    sts128(stg + stg_off(lane, q), w);
  }
}
// lane = row: 32 fp32 as bf16 into a 32 x 64 B tile in the TMA SWIZZLE_64B image (16-byte piece q of row r at
// r * 64 + ((q ^ ((r >> 1) & 3)) << 4)): what a bulk tensor store with a {32 columns, 32 rows} box reads; conflict-free
__device__ __forceinline__ void stg_put_row_sw64(uint32_t stg, int lane, const float (&v)[32]) {
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    uint4 w;
    w.x = pack_bf16x2(v[q * 8 + 0], v[q * 8 + 1]);
    w.y = pack_bf16x2(v[q * 8 + 2], v[q * 8 + 3]);
    w.z = pack_bf16x2(v[q * 8 + 4], v[q * 8 + 5]);
    w.w = pack_bf16x2(v[q * 8 + 6], v[q * 8 + 7]);
    sts128(stg + lane * 64 + ((q ^ ((lane >> 1) & 3)) << 4), w);
  }
}
// whole warp: staging tile -> global rows [0, rows_valid) x 32 columns at g (row stride ld elements); 4 lanes per row
__device__ __forceinline__ void stg_to_global(uint32_t stg, bf16* g, size_t ld, int lane, int rows_valid) {
  uint4 w[4];
#pragma unroll
  for (int it = 0; it < 4; ++it) w[it] = lds128(stg + stg_off(it * 8 + (lane >> 2), lane & 3));
#pragma unroll
  for (int it = 0; it < 4; ++it) {
    const int r = it * 8 + (lane >> 2), c = lane & 3;
    if (r < rows_valid) *reinterpret_cast<uint4*>(g + (size_t)r * ld + c * 8) = w[it];
  }
}

// instruction descriptor: D fp32, A/B bf16, M = 256 (pair), N = n, majorness per operand (0 = K-major, 1 = MN-major)
__host__ __device__ constexpr uint32_t make_idesc(int a_mn, int b_mn, int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_mn << 15) | ((uint32_t)b_mn << 16) | ((uint32_t)(n >> 3) << 17) |
         ((uint32_t)((2 * BM) >> 4) << 24);
}

// ---------------------------------------------------------------------------------------------------------
// tile decode shared by the three roles (identical in both CTAs of a pair except for the rank-dependent fields)
// ---------------------------------------------------------------------------------------------------------
struct Tile {
  int row0;        // first of THIS CTA's 128 rows (row modes) / output rows (WGRAD)
  bool live;       // this CTA's rows exist (false: second half of a single-tile pair, or beyond the row count)
  bool peer_live;  // row modes: CTA 1's rows exist
  int n_tile;      // column tile
  int n_mma;       // N of the MMA: 256, or 128 when at most 128 columns of the tile exist
  int slot, part, group;  // group: WGRAD only
  int num_kb;      // 64-wide K blocks
  int k_row0;      // WGRAD: first row of the K range
  int job;         // WGRAD: job index (0 when the launch has a single weight gradient)
  int M, N;        // WGRAD: output extent of the job
  int a_gcol, b_gcol;  // WGRAD: per-group column offsets of the job's operands
  int piece;       // WGRAD tail split: index of this K piece in tail_part, -1 = a whole tile
};

template <int MODE>
struct Sched {
  const UmmaParams& p;
  const int rank;
  int n_tiles_n, ntn_total, m_pairs;
  long total;
  __device__ Sched(const UmmaParams& p_, int rank_) : p(p_), rank(rank_) {
    const bool dense = p.n_mtiles == nullptr;
    if (MODE == WGRAD) {
      m_pairs = (p.M + 2 * BM - 1) / (2 * BM);
      n_tiles_n = (p.N + BN - 1) / BN;
      ntn_total = n_tiles_n;
      total = (long)p.n_groups * m_pairs * n_tiles_n;
      if (p.tail_ks > 1) total = p.tail_first + (total - p.tail_first) * p.tail_ks;
      if (p.n_jobs > 0) {
        total = 0;
        for (int j = 0; j < p.n_jobs; ++j)
          total += (long)p.n_groups * ((p.job_M[j] + 2 * BM - 1) / (2 * BM)) * ((p.job_N[j] + BN - 1) / BN);
      }
    } else {
      m_pairs = dense ? (p.dense_rows + 2 * BM - 1) / (2 * BM) : p.n_mtiles[2];
      const int n_extent = (MODE == FWD1 || MODE == FWD1S || MODE == DH) ? p.F : p.d;
      const int bn = MODE == FWD1 ? BN / 2 : BN;
      n_tiles_n = MODE == ROUTE ? 1 : (n_extent + bn - 1) / bn;
      ntn_total = n_tiles_n * ((dense && (MODE == FWD1 || MODE == FWD1S || MODE == DH)) ? p.parts : 1);
      total = (long)m_pairs * ntn_total;
    }
  }
  __device__ Tile decode(long id) const {
    Tile t;
    const bool dense = p.n_mtiles == nullptr;
    if (MODE == WGRAD) {
      t.piece = -1;
      int kpart = 0;
      if (p.tail_ks > 1 && id >= p.tail_first) {
        t.piece = (int)(id - p.tail_first);
        kpart = t.piece % p.tail_ks;
        id = p.tail_first + t.piece / p.tail_ks;
      }
      int mp = m_pairs, ntn = n_tiles_n;
      t.job = 0; t.M = p.M; t.N = p.N; t.a_gcol = p.a_gcol; t.b_gcol = p.b_gcol;
      for (int j = 0; j < p.n_jobs; ++j) {      // which job: tiles are numbered job after job
        t.job = j; t.M = p.job_M[j]; t.N = p.job_N[j]; t.a_gcol = p.job_agcol[j]; t.b_gcol = p.job_bgcol[j];
        mp = (t.M + 2 * BM - 1) / (2 * BM);
        ntn = (t.N + BN - 1) / BN;
        const long nj = (long)p.n_groups * mp * ntn;
        if (id < nj) break;
        id -= nj;
      }
      t.group = (int)(id / ((long)mp * ntn));
      int rem = (int)(id % ((long)mp * ntn));
      t.row0 = (rem / ntn) * 2 * BM + rank * BM;
      t.live = t.row0 < t.M;
      t.peer_live = true;
      t.n_tile = rem % ntn;
      t.n_mma = (t.N - t.n_tile * BN <= BN / 2) ? BN / 2 : BN;
      t.slot = t.part = t.group;
      int r0, r1;
      if (p.pad_offsets) { r0 = p.pad_offsets[t.group]; r1 = p.pad_end64[t.group]; }
      else if (p.k_chunk > 0) { r0 = min(t.group * p.k_chunk, p.dense_rows); r1 = min(r0 + p.k_chunk, p.dense_rows); }
      else { r0 = 0; r1 = p.dense_rows; }
      if (t.piece >= 0) { r0 = min(kpart * p.tail_chunk, p.dense_rows); r1 = min(r0 + p.tail_chunk, p.dense_rows); }
      t.k_row0 = r0;
      t.num_kb = (r1 - r0 + BK - 1) / BK;
    } else {
      const int pair = (int)(id / ntn_total);
      int nidx = (int)(id % ntn_total);
      t.part = nidx / n_tiles_n;
      t.n_tile = nidx % n_tiles_n;
      if (dense) {
        t.row0 = pair * 2 * BM + rank * BM;
        t.live = t.row0 < p.dense_rows;
        t.peer_live = pair * 2 * BM + BM < p.dense_rows;
        t.slot = t.part;
      } else {
        const int info = p.pair_info[pair];
        const int first = info >> 1;
        t.row0 = (first + rank) * BM;
        t.live = rank == 0 || (info & 1);
        t.peer_live = (info & 1) != 0;
        t.slot = p.tile_slot[first];
      }
      t.group = 0;
      t.k_row0 = 0;
      const int kparts = dense ? p.parts : 1;
      const int n_extent = (MODE == DH || MODE == FWD1S) ? p.F : p.d;
      t.n_mma = MODE == ROUTE ? p.N : (MODE != FWD1 && n_extent - t.n_tile * BN <= BN / 2) ? BN / 2 : BN;
      if (MODE == FWD1 || MODE == FWD1S || MODE == DH || MODE == ROUTE) t.num_kb = p.d / BK;
      else if (MODE == FWD2) t.num_kb = kparts * (p.F / BK);
      else t.num_kb = p.ksegs * kparts * (p.F / BK);  // DX
    }
    return t;
  }
};

// ---------------------------------------------------------------------------------------------------------
// ROUTE epilogue: gate + top-k + residency mask + per-block histogram straight from tensor memory.
// Accumulator columns are [hi | mid | lo] pieces of the logits (Epad columns each, see route_umma.cu); a token row is one
// TMEM lane.  Two warps share a lane quarter: warp `half` takes the 16-expert chunks half, half + 2, ...; they exchange
// their partial max / top-k list / softmax sum through shared memory (named barrier 1 + q, 64 threads) and the
// half-0 thread finishes the token.  Selection is on the logits z (ties -> lower expert id), Eq. 14;
// mask and gate rule PAPER.md:157-159, 593.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
  uint32_t* r = reinterpret_cast<uint32_t*>(v);
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                 "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr));
}
__device__ __forceinline__ void bar_sync_named(int id, int threads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory"); }

constexpr int kNetK = 16;     // largest top-k list the sorting-network epilogue handles (k <= 16); k = 17..32 takes the insertion epilogue
template <int KMAX>
struct RouteSmem {            // lives in the kernel's staging area (route_stg_bytes(KMAX) bytes)
  static constexpr int KN = KMAX > kNetK ? kNetK : (KMAX < 2 ? 2 : KMAX);   // capacity of the sorting-network lists
  static constexpr int KI = KMAX > kNetK ? KMAX : 1;                          // capacity of the insertion lists
  int32_t slot[128];          // resident slot of expert e, -1 = ghost
  float zb[128];              // additive logit term of expert e: router bias (or 0); -inf = no such column (e >= E, or a ghost
                              // expert under forced-local routing)
  int32_t hist[kAccStages][128];
  float mx[2][128];           // partial max of each half
  float sum[2][128];          // partial softmax denominators
  union {
    struct {                  // insertion epilogue (k > kNetK)
      float lv[KI][128];      // half 1 -> half 0: top-k values / ids of row r
      int32_t li[KI][128];
    } ins;
    struct {                  // sorting-network epilogue
      uint2 hand[KN][128];             // half 1 -> half 0: sorted (value, id) list of row r
      uint2 cand[KN + 1][256];         // per-thread candidate lists (thread-private), written in id order
    } net;
  };
};
static_assert(sizeof(RouteSmem<2>) <= route_stg_bytes(2) && sizeof(RouteSmem<4>) <= route_stg_bytes(4) &&
              sizeof(RouteSmem<8>) <= route_stg_bytes(8) && sizeof(RouteSmem<16>) <= route_stg_bytes(16) &&
              sizeof(RouteSmem<32>) <= route_stg_bytes(32), "route epilogue scratch");
static_assert(smem_bytes_of(ROUTE, 8) <= 227 * 1024 && smem_bytes_of(ROUTE, 16) <= 227 * 1024 && smem_bytes_of(ROUTE, 32) <= 227 * 1024, "shared memory");

// ---- sorting networks on registers (all indices are compile-time: nothing spills) ----
// Descending bitonic networks.  Values only: a compare-exchange is one FMNMX pair; a NaN operand is dropped by fmaxf / fminf
// (the other operand is duplicated), which can only RAISE the outputs.
template <int N> struct NetV {
  static __device__ __forceinline__ void ce(float& a, float& b) { const float hi = fmaxf(a, b), lo = fminf(a, b); a = hi; b = lo; }
  static __device__ __forceinline__ void merge(float (&v)[N]) {   // bitonic sequence -> descending
#pragma unroll
    for (int j = N >> 1; j > 0; j >>= 1)
#pragma unroll
      for (int i = 0; i < N; ++i)
        if ((i ^ j) > i) ce(v[i], v[i ^ j]);
  }
  static __device__ __forceinline__ void sort(float (&v)[N]) {
#pragma unroll
    for (int k = 2; k <= N; k <<= 1)
#pragma unroll
      for (int j = k >> 1; j > 0; j >>= 1)
#pragma unroll
        for (int i = 0; i < N; ++i)
          if ((i ^ j) > i) { if ((i & k) == 0) ce(v[i], v[i ^ j]); else ce(v[i ^ j], v[i]); }
  }
};
// (value, id) pairs in the order of PAPER.md:519 Eq. 14 as read in DESIGN.md R5: larger logit first, ties -> lower expert id
template <int N> struct NetKV {
  static __device__ __forceinline__ void ce(float& av, int& ai, float& bv, int& bi) {   // afterwards a comes before b
    const bool sw = bv > av || (bv == av && bi < ai);
    const float v = sw ? bv : av, w = sw ? av : bv;
    const int i = sw ? bi : ai, j = sw ? ai : bi;
    av = v; bv = w; ai = i; bi = j;
  }
  static __device__ __forceinline__ void merge(float (&v)[N], int (&id)[N]) {
#pragma unroll
    for (int j = N >> 1; j > 0; j >>= 1)
#pragma unroll
      for (int i = 0; i < N; ++i)
        if ((i ^ j) > i) ce(v[i], id[i], v[i ^ j], id[i ^ j]);
  }
  static __device__ __forceinline__ void sort(float (&v)[N], int (&id)[N]) {
#pragma unroll
    for (int k = 2; k <= N; k <<= 1)
#pragma unroll
      for (int j = k >> 1; j > 0; j >>= 1)
#pragma unroll
        for (int i = 0; i < N; ++i)
          if ((i ^ j) > i) { if ((i & k) == 0) ce(v[i], id[i], v[i ^ j], id[i ^ j]); else ce(v[i ^ j], id[i ^ j], v[i], id[i]); }
  }
};
__device__ __forceinline__ void sts64(uint32_t addr, uint32_t a, uint32_t b) {
  asm volatile("st.shared.v2.b32 [%0], {%1, %2};" ::"r"(addr), "r"(a), "r"(b) : "memory");
}
__device__ __forceinline__ uint2 lds64(uint32_t addr) {
  uint2 v;
  asm volatile("ld.shared.v2.b32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void stg256(float* p, const float* v) {   // 32-byte store: one whole sector per lane
  asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]), "f"(v[4]),
               "f"(v[5]), "f"(v[6]), "f"(v[7]) : "memory");
}

// Sorting-network ROUTE epilogue (k <= kNetK).  A thread owns one token row and, of its experts, the 16-wide chunks half,
// half + 2, ...  Selection without data-dependent branches (a per-lane insertion list makes every lane pay for every
// insertion of any lane, in one long dependent chain), in three rolled passes over the thread's chunks -- each pass re-reads
// the chunk from tensor memory and recombines it with the SAME instruction sequence, so the values are bit-identical (small
// code: the unrolled single-pass form overflowed the instruction cache and spilled):
//   A. top-KMAX VALUES by bitonic networks of FMNMX (groups of KMAX sorted, merged into the running list);
//   B. the KMAX-th value is the threshold: logits above it, and the first ones equal to it in id order, are the candidates
//      -- written with predicated stores to a thread-private list in shared memory (exactly the top KMAX, ties -> lower id);
//      the same pass sums exp(z - local max) for the softmax;
//      then the <= KMAX candidates are sorted with their ids and the two halves' lists merged by half 0;
//   C. probabilities.
template <int KMAX>
__device__ __forceinline__ void route_tile_epilogue_net(const UmmaParams& p, RouteSmem<KMAX>* rs, uint32_t taddr, int q, int half, int lane, int as,
                                                        int row0, bool live) {
  const RouteEpi& r = p.r;
  const int E = r.E, Epad = r.Epad;
  const bool three = r.pieces == 3, softmax = r.gate_fn == FOMOE_GATE_SOFTMAX;
  const int rl = q * 32 + lane;        // row within the CTA's 128
  const int t = row0 + rl;
  const bool row_ok = live && t < p.dense_rows;
  if (live) {
    auto load_z = [&](int c0, float (&z)[16]) {   // logits of 16 experts from c0: identical arithmetic in every pass
      float md[16], lo[16];
      tmem_ld16(taddr + c0, z);
      tmem_ld16(taddr + Epad + c0, md);
      if (three) tmem_ld16(taddr + 2 * Epad + c0, lo);
      float zb[16];
#pragma unroll
      for (int v = 0; v < 4; ++v) *reinterpret_cast<float4*>(&zb[4 * v]) = *reinterpret_cast<const float4*>(&rs->zb[c0 + 4 * v]);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        float sacc = __fadd_rn(z[i], md[i]);
        if (three) sacc = __fadd_rn(sacc, lo[i]);
        z[i] = __fmaf_rn(sacc, r.inv_tau, zb[i]);   // (padding columns of the accumulator are exactly 0: 0 * inv_tau - inf = -inf)
      }
    };
    // A. top-KMAX values, descending
    float tv[KMAX];
#pragma unroll
    for (int j = 0; j < KMAX; ++j) tv[j] = -INFINITY;
#pragma unroll 1
    for (int c0 = 16 * half; c0 < Epad; c0 += 32) {
      float z[16];
      load_z(c0, z);
#pragma unroll
      for (int g = 0; g < 16 / KMAX; ++g) {
        float sv[KMAX];
#pragma unroll
        for (int j = 0; j < KMAX; ++j) sv[j] = z[g * KMAX + j];
        NetV<KMAX>::sort(sv);
#pragma unroll
        for (int j = 0; j < KMAX; ++j) tv[j] = fmaxf(tv[j], sv[KMAX - 1 - j]);   // the top half of the 2 KMAX values, bitonic
        NetV<KMAX>::merge(tv);
      }
    }
    const float mxl = tv[0];
    const float mxe = mxl == -INFINITY ? 0.f : mxl;   // (no finite logit in this half: every exponential below is exp(-inf) = 0)
    rs->mx[half][rl] = mxl;
    // B. candidates: > threshold, and the first `need` ones == threshold; softmax partial sum against the local max
    const float thr = tv[KMAX - 1];
    int need = KMAX;
#pragma unroll
    for (int j = 0; j < KMAX - 1; ++j) need -= tv[j] > thr ? 1 : 0;
    const uint32_t cand0 = smem_u32(&rs->net.cand[0][half * 128 + rl]);
    constexpr uint32_t kCandStride = 256 * sizeof(uint2);
#pragma unroll
    for (int j = 0; j < KMAX; ++j) sts64(cand0 + j * kCandStride, __float_as_uint(-INFINITY), (uint32_t)kMaxE);
    float sml = 0.f;
    {
      uint32_t ca = cand0;
      int eqc = 0;
#pragma unroll 1
      for (int c0 = 16 * half; c0 < Epad; c0 += 32) {
        float z[16];
        load_z(c0, z);
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const float v = z[i];
          const bool eq = v == thr && eqc < need;
          if (v > thr || eq) { sts64(ca, __float_as_uint(v), (uint32_t)(c0 + i)); ca += kCandStride; }
          eqc += eq ? 1 : 0;
        }
        if (softmax) {
#pragma unroll
          for (int i = 0; i < 16; ++i) sml += __expf(z[i] - mxe);   // (exp(-inf) = 0 for the columns that do not exist)
        }
      }
    }
    rs->sum[half][rl] = sml;
    float cv[KMAX];
    int ci[KMAX];
#pragma unroll
    for (int j = 0; j < KMAX; ++j) {
      const uint2 e = lds64(cand0 + j * kCandStride);
      cv[j] = __uint_as_float(e.x);
      ci[j] = (int)e.y;
    }
    NetKV<KMAX>::sort(cv, ci);
    if (half == 1) {
#pragma unroll
      for (int j = 0; j < KMAX; ++j) rs->net.hand[j][rl] = make_uint2(__float_as_uint(cv[j]), (uint32_t)ci[j]);
    }
    bar_sync_named(1 + q, 64);
    const float mx0 = rs->mx[0][rl], mx1 = rs->mx[1][rl];
    const float mx = fmaxf(mx0, mx1);
    float inv_s = 1.f;
    if (softmax) {   // denominators of the two halves, rescaled to the common max (a half without experts: max -inf, sum 0)
      const float s0 = rs->sum[0][rl], s1 = rs->sum[1][rl];
      inv_s = 1.0f / ((mx0 == mx || s0 == 0.f ? s0 : s0 * __expf(mx0 - mx)) + (mx1 == mx || s1 == 0.f ? s1 : s1 * __expf(mx1 - mx)));
    }
    if (half == 0) {   // top KMAX of the two sorted lists: pairwise "earlier of a[j], b[KMAX-1-j]" is bitonic, then merge
#pragma unroll
      for (int j = 0; j < KMAX; ++j) {
        const uint2 e = rs->net.hand[KMAX - 1 - j][rl];
        const float bv = __uint_as_float(e.x);
        const int bi = (int)e.y;
        const bool sw = bv > cv[j] || (bv == cv[j] && bi < ci[j]);
        cv[j] = sw ? bv : cv[j];
        ci[j] = sw ? bi : ci[j];
      }
      NetKV<KMAX>::merge(cv, ci);
      // fewer than k logits compare greater than -inf (NaN / inf activations, a -inf bias): the list still holds the sentinel id.
      // Keep every id in range so that neither the slot lookup below nor the permutation kernels index with it
#pragma unroll
      for (int j = 0; j < KMAX; ++j) ci[j] = min(ci[j], E - 1);
    }
    auto prob_of = [&](float zz) { return softmax ? __expf(zz - mx) * inv_s : __fdividef(1.0f, 1.0f + __expf(-zz)); };
    // C. probabilities of this warp's chunks
#pragma unroll 1
    for (int c0 = 16 * half; c0 < Epad; c0 += 32) {
      float z[16];
      load_z(c0, z);
#pragma unroll
      for (int i = 0; i < 16; ++i) z[i] = prob_of(z[i]);
      if (row_ok) {
        float* dst = r.probs + (size_t)t * E + c0;
        if ((E & 7) == 0) {
          if (c0 < E) stg256(dst, &z[0]);
          if (c0 + 8 < E) stg256(dst + 8, &z[8]);
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i)
            if (c0 + i < E) dst[i] = z[i];
        }
      }
    }
    // residency mask, gate rule, outputs, per-slot histogram of the block
    if (half == 0 && row_ok) {
      float pj[KMAX];
      int sl[KMAX];
      float s_all = 0.f, s_kept = 0.f;
#pragma unroll
      for (int j = 0; j < KMAX; ++j) {
        pj[j] = 0.f;
        sl[j] = -1;
        if (j < r.k) {
          pj[j] = prob_of(cv[j]);
          sl[j] = rs->slot[ci[j]];
          s_all += pj[j];
          if (sl[j] >= 0) s_kept += pj[j];
        }
      }
#pragma unroll
      for (int j = 0; j < KMAX; ++j) {
        if (j < r.k) {
          float g = 0.f;
          if (sl[j] >= 0) {
            g = r.gate_rule == FOMOE_DROP_ONLY ? pj[j] : r.gate_rule == FOMOE_RENORM_TOPK ? pj[j] / s_all : pj[j] / s_kept;
            atomicAdd(&rs->hist[as][sl[j]], 1);
          }
          r.topk_idx[(size_t)t * r.k + j] = ci[j];
          r.gate[(size_t)t * r.k + j] = g;
        }
      }
    }
  }
  // all 8 epilogue warps: the block's histogram is complete; flush and clear it (next use of hist[as] is two tiles later)
  bar_sync_named(5, kEpiWarps * 32);
  if (live) {
    const int tid = (half * 4 + q) * 32 + lane;
    for (int i = tid; i < r.n_res; i += kEpiWarps * 32) {
      r.blk_hist[(size_t)(row0 / BM) * r.n_res + i] = rs->hist[as][i];
      rs->hist[as][i] = 0;
    }
  }
}

template <int KMAX>
__device__ __forceinline__ void route_tile_epilogue(const UmmaParams& p, RouteSmem<KMAX>* rs, uint32_t taddr, int q, int half, int lane, int as,
                                                    int row0, bool live) {
  const RouteEpi& r = p.r;
  const int E = r.E, Epad = r.Epad;
  const bool three = r.pieces == 3, softmax = r.gate_fn == FOMOE_GATE_SOFTMAX;
  const int rl = q * 32 + lane;        // row within the CTA's 128
  const int t = row0 + rl;
  const bool row_ok = live && t < p.dense_rows;
  if (live) {
    auto load_z = [&](int c0, float (&z)[16]) {   // logits of 16 experts from c0: identical arithmetic in every pass
      float md[16], lo[16];
      tmem_ld16(taddr + c0, z);
      tmem_ld16(taddr + Epad + c0, md);
      if (three) tmem_ld16(taddr + 2 * Epad + c0, lo);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        float s = z[i] + md[i];
        if (three) s += lo[i];
        z[i] = s * r.inv_tau + (r.bias && c0 + i < E ? r.bias[c0 + i] : 0.f);
        // forced-local routing: no router column for a non-resident expert: logit -inf, probability 0
        if (r.forced_local && c0 + i < E && rs->slot[c0 + i] < 0) z[i] = -INFINITY;
      }
    };
    // pass 1: partial max and partial top-KMAX (descending, ties -> lower id: ascending scan + strict '>')
    float tv[KMAX];
    int ti[KMAX];
#pragma unroll
    for (int j = 0; j < KMAX; ++j) { tv[j] = -INFINITY; ti[j] = kMaxE; }
    float mx = -INFINITY;
#pragma unroll 1
    for (int c0 = 16 * half; c0 < Epad; c0 += 32) {
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
    rs->mx[half][rl] = mx;
    if (half == 1) {
#pragma unroll
      for (int j = 0; j < KMAX; ++j) { rs->ins.lv[j][rl] = tv[j]; rs->ins.li[j][rl] = ti[j]; }
    }
    bar_sync_named(1 + q, 64);
    mx = fmaxf(rs->mx[0][rl], rs->mx[1][rl]);
    if (half == 0) {   // merge the partner's list: insert its entries (descending) with the (value, lower id) order
#pragma unroll 1
      for (int jj = 0; jj < KMAX; ++jj) {
        float cv = rs->ins.lv[jj][rl];
        int ci = rs->ins.li[jj][rl];
        bool ins = false;
#pragma unroll
        for (int j = 0; j < KMAX; ++j) {
          const bool gt = ins || cv > tv[j] || (cv == tv[j] && ci < ti[j]);
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
    // fewer than k logits compare greater than -inf (NaN / inf activations, a -inf bias): the list still holds the sentinel id.
    // Keep every id in range so that neither the slot lookup below nor the permutation kernels index with it
    if (half == 0) {
#pragma unroll
      for (int j = 0; j < KMAX; ++j) ti[j] = min(ti[j], E - 1);
    }
    // pass 2 (softmax): denominator, summed as (half 0) + (half 1) by both warps
    float inv_s = 1.f;
    if (softmax) {
      float sm = 0.f;
  #pragma unroll 1
    for (int c0 = 16 * half; c0 < Epad; c0 += 32) {
        float z[16];
        load_z(c0, z);
#pragma unroll
        for (int i = 0; i < 16; ++i)
          if (c0 + i < E) sm += __expf(z[i] - mx);
      }
      rs->sum[half][rl] = sm;
      bar_sync_named(1 + q, 64);
      inv_s = 1.0f / (rs->sum[0][rl] + rs->sum[1][rl]);
    }
    auto prob_of = [&](float z) { return softmax ? __expf(z - mx) * inv_s : __fdividef(1.0f, 1.0f + __expf(-z)); };
    // pass 3: probabilities of this warp's chunks
#pragma unroll 1
    for (int c0 = 16 * half; c0 < Epad; c0 += 32) {
      float z[16];
      load_z(c0, z);
#pragma unroll
      for (int i = 0; i < 16; ++i) z[i] = prob_of(z[i]);
      if (row_ok) {
        float* dst = r.probs + (size_t)t * E + c0;
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
    // residency mask, gate rule, outputs, per-slot histogram of the block
    if (half == 0 && row_ok) {
      float pj[KMAX];
      int sl[KMAX];
      float s_all = 0.f, s_kept = 0.f;
#pragma unroll
      for (int j = 0; j < KMAX; ++j) {
        pj[j] = 0.f;
        sl[j] = -1;
        if (j < r.k) {
          pj[j] = prob_of(tv[j]);
          sl[j] = rs->slot[ti[j]];
          s_all += pj[j];
          if (sl[j] >= 0) s_kept += pj[j];
        }
      }
#pragma unroll
      for (int j = 0; j < KMAX; ++j) {
        if (j < r.k) {
          float g = 0.f;
          if (sl[j] >= 0) {
            g = r.gate_rule == FOMOE_DROP_ONLY ? pj[j] : r.gate_rule == FOMOE_RENORM_TOPK ? pj[j] / s_all : pj[j] / s_kept;
            atomicAdd(&rs->hist[as][sl[j]], 1);
          }
          r.topk_idx[(size_t)t * r.k + j] = ti[j];
          r.gate[(size_t)t * r.k + j] = g;
        }
      }
    }
  }
  // all 8 epilogue warps: the block's histogram is complete; flush and clear it (next use of hist[as] is two tiles later)
  bar_sync_named(5, kEpiWarps * 32);
  if (live) {
    const int tid = (half * 4 + q) * 32 + lane;
    for (int i = tid; i < r.n_res; i += kEpiWarps * 32) {
      r.blk_hist[(size_t)(row0 / BM) * r.n_res + i] = rs->hist[as][i];
      rs->hist[as][i] = 0;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------------------
template <int MODE, int KMAX = 0>   // KMAX: ROUTE only, capacity of the top-k list (2, 4, 8, 16 or 32)
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
umma_grouped_kernel(const __grid_constant__ TmaMaps maps, const __grid_constant__ UmmaParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  constexpr int kStages = stages_of(MODE, KMAX);
  constexpr int kStgTilesPerWarp = stg_tiles_per_warp(MODE);
  uint8_t* stg_base = smem + kStages * kStageBytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(stg_base + stg_bytes_of(MODE, KMAX));
  uint64_t* full_bar = bars;                          // [kStages]   used in the leader CTA only
  uint64_t* empty_bar = bars + kStages;               // [kStages]   one per CTA, released by the leader's commits
  uint64_t* tfull_bar = bars + 2 * kStages;           // [kAccStages] one per CTA
  uint64_t* tempty_bar = bars + 2 * kStages + kAccStages;  // [kAccStages] leader only: 8 epilogue warps x 2 CTAs
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * kStages + 2 * kAccStages);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int rank = (int)cluster_ctarank();
  const int cluster_id = blockIdx.x >> 1, n_clusters = gridDim.x >> 1;
  constexpr bool kAMn = (MODE == WGRAD), kBMn = (MODE == DH || MODE == DX || MODE == WGRAD || MODE == ROUTE);

  pdl_launch_dependents();
  if (warp == 0 && lane == 0) {
#pragma unroll
    for (int i = 0; i < 4; ++i) prefetch_tmap(&maps.m[i]);
    if (MODE == WGRAD && p.n_jobs > 2) { prefetch_tmap(&maps.m[4]); prefetch_tmap(&maps.m[5]); }   // (zero-filled otherwise)
    if ((MODE == FWD2 || MODE == DX) && p.tma_store) prefetch_tmap(&maps.m[4]);
    if ((MODE == FWD1 || MODE == FWD1S) && p.tma_store) { prefetch_tmap(&maps.m[3]); prefetch_tmap(&maps.m[5]); if (MODE == FWD1) prefetch_tmap(&maps.m[4]); }
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < kStages; ++i) { mbar_init(smem_u32(&full_bar[i]), 1); mbar_init(smem_u32(&empty_bar[i]), 1); }
    for (int i = 0; i < kAccStages; ++i) { mbar_init(smem_u32(&tfull_bar[i]), 1); mbar_init(smem_u32(&tempty_bar[i]), 2 * kEpiWarps); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(kTmemCols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  cluster_sync_all();   // barriers of both CTAs initialised, tensor memory allocated in both
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  pdl_wait();   // the prologue above touched only shared / tensor memory; everything below reads the previous kernels' output

  const Sched<MODE> sched(p, rank);
  const bool dense = p.n_mtiles == nullptr;

  if (warp == 0) {
    // ===================== TMA producer (both CTAs; completion bytes land on the leader's barrier) =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (long id = cluster_id; id < sched.total; id += n_clusters) {
        const Tile t = sched.decode(id);
        const int m0 = t.row0;
        const int nh = t.n_mma / 2;                 // B columns staged by each CTA
        const bool peer_live = MODE == WGRAD || t.peer_live;
        for (int kb = 0; kb < t.num_kb; ++kb) {
          mbar_wait(smem_u32(&empty_bar[stage]), phase ^ 1);
          const uint32_t sa = smem_u32(smem + stage * kStageBytes), sb = sa + kABytes;
          const uint32_t fb = smem_u32(&full_bar[stage]) & 0xFEFFFFFFu;   // peer bit cleared: the pair leader's barrier
          // a pair whose second row tile does not exist (odd tile count of a slot, or the dense tail) skips CTA 1's A load:
          // the MMA then reads stale shared memory for rows nobody stores.  `peer_live` is what CTA 1 decodes as t.live
          if (rank == 0) mbar_expect_tx(smem_u32(&full_bar[stage]), 2 * kStageBytes - (peer_live ? 0 : kABytes));
          if (MODE == FWD1) {
            if (t.live) tma_load_2d_2sm(sa, &maps.m[0], fb, kb * BK, m0);
            // N columns [0,128) = a (W_gate rows, staged by CTA 0), [128,256) = u (W_up rows, CTA 1)
            tma_load_2d_2sm(sb, &maps.m[1 + rank], fb, kb * BK, t.slot * p.F + t.n_tile * (BN / 2));
          } else if (MODE == FWD1S) {   // B = W_up rows [slot F + n_tile BN + rank nh, ..), K-major
            if (t.live) tma_load_2d_2sm(sa, &maps.m[0], fb, kb * BK, m0);
            tma_load_2d_2sm(sb, &maps.m[1], fb, kb * BK, t.slot * p.F + t.n_tile * BN + rank * nh);
          } else if (MODE == FWD2) {
            const int kpp = p.F / BK, part = kb / kpp, kk = kb % kpp;
            if (t.live) tma_load_2d_2sm(sa, &maps.m[0], fb, part * p.F + kk * BK, m0);
            tma_load_2d_2sm(sb, &maps.m[1], fb, kk * BK, (dense ? part : t.slot) * p.d + t.n_tile * BN + rank * nh);
          } else if (MODE == ROUTE) {   // A = x rows (K-major), B = split W_r [d, N] (MN-major), CTA r stages columns [r N/2, (r+1) N/2)
            if (t.live) tma_load_2d_2sm(sa, &maps.m[0], fb, kb * BK, m0);
#pragma unroll
            for (int j = 0; j < BN / 128; ++j) tma_load_2d_2sm(sb + j * 8192, &maps.m[1], fb, rank * nh + 64 * j, kb * BK);
          } else if (MODE == DH) {
            if (t.live) tma_load_2d_2sm(sa, &maps.m[0], fb, kb * BK, m0);
#pragma unroll
            for (int j = 0; j < BN / 128; ++j)
              tma_load_2d_2sm(sb + j * 8192, &maps.m[1], fb, t.n_tile * BN + rank * nh + 64 * j, t.slot * p.d + kb * BK);
          } else if (MODE == DX) {
            const int kseg = (dense ? p.parts : 1) * (p.F / BK), seg = kb / kseg, kk = kb % kseg;
            if (t.live) tma_load_2d_2sm(sa, &maps.m[seg], fb, kk * BK, m0);
            const int brow = (dense ? 0 : t.slot * p.F) + kk * BK;
#pragma unroll
            for (int j = 0; j < BN / 128; ++j)
              tma_load_2d_2sm(sb + j * 8192, &maps.m[2 + seg], fb, t.n_tile * BN + rank * nh + 64 * j, brow);
          } else {  // WGRAD
            const int r = t.k_row0 + kb * BK;
#pragma unroll
            for (int i = 0; i < BM / 64; ++i) tma_load_2d_2sm(sa + i * 8192, &maps.m[2 * t.job], fb, t.group * t.a_gcol + m0 + 64 * i, r);
#pragma unroll
            for (int j = 0; j < BN / 128; ++j)
              tma_load_2d_2sm(sb + j * 8192, &maps.m[2 * t.job + 1], fb, t.group * t.b_gcol + t.n_tile * BN + rank * nh + 64 * j, r);
          }
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA) =====================
    // The whole warp walks the (warp-uniform) schedule and waits on the barriers; one elected lane issues.  What bounds
    // this loop is the issuing thread's own instruction latency per MMA, so the per-stage descriptor words are
    // precomputed (lane s holds stage s, fetched with one shuffle) and a K step is one 32-bit add.
    if (rank == 0) {
      int stage = 0, as = 0;
      uint32_t phase = 0, aphase = 0;
      // K-major: 16 K-elements = 32 bytes inside the 128-byte swizzle row, row groups 1024 B apart.
      // MN-major: 16 K-rows = two 8-row swizzle atoms (2 x 1024 B); 64-element MN chunks 8192 B apart.
      const uint32_t sa0 = smem_u32(smem) + (uint32_t)(lane < kStages ? lane : 0) * kStageBytes, sb0 = sa0 + kABytes;
      const uint64_t adesc_l = kAMn ? make_desc(sa0, 8192, 1024) : make_desc(sa0, 16, 1024);
      const uint64_t bdesc_l = kBMn ? make_desc(sb0, 8192, 1024) : make_desc(sb0, 16, 1024);
      const uint32_t a_hi = (uint32_t)(adesc_l >> 32), b_hi = (uint32_t)(bdesc_l >> 32);
      const uint32_t my_alo = (uint32_t)adesc_l, my_blo = (uint32_t)bdesc_l;
      constexpr uint32_t kAStep = (kAMn ? 2048 : 32) >> 4, kBStep = (kBMn ? 2048 : 32) >> 4;
      for (long id = cluster_id; id < sched.total; id += n_clusters) {
        const Tile t = sched.decode(id);
        if (t.num_kb == 0) continue;  // empty WGRAD group: the epilogue writes zeros without touching TMEM
        const uint32_t idesc = make_idesc(kAMn ? 1 : 0, kBMn ? 1 : 0, t.n_mma);
        mbar_wait(smem_u32(&tempty_bar[as]), aphase ^ 1);
        const uint32_t tmem_d = tmem_base + as * BN;
        const int num_kb = t.num_kb;
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(smem_u32(&full_bar[stage]), phase);
          tc_fence_after();
          const uint32_t alo = __shfl_sync(0xffffffffu, my_alo, stage), blo = __shfl_sync(0xffffffffu, my_blo, stage);
          if (elect_one_sync()) {
            umma_bf16_2sm_lohi(tmem_d, alo, a_hi, blo, b_hi, idesc, kb != 0 ? 1u : 0u);
            umma_bf16_2sm_lohi(tmem_d, alo + kAStep, a_hi, blo + kBStep, b_hi, idesc, 1u);
            umma_bf16_2sm_lohi(tmem_d, alo + 2 * kAStep, a_hi, blo + 2 * kBStep, b_hi, idesc, 1u);
            umma_bf16_2sm_lohi(tmem_d, alo + 3 * kAStep, a_hi, blo + 3 * kBStep, b_hi, idesc, 1u);
            umma_commit_2sm(smem_u32(&empty_bar[stage]), 3);                    // frees the stage in both CTAs
            if (kb == num_kb - 1) umma_commit_2sm(smem_u32(&tfull_bar[as]), 3);  // accumulator complete, both CTAs
          }
          __syncwarp();
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        if (++as == kAccStages) { as = 0; aphase ^= 1; }
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue (each CTA drains its own 128 accumulator rows) =====================
    const int q = warp & 3;               // TMEM lane quarter of this warp
    const int half = (warp >> 2) - 1;     // which of the two warps of the quarter: takes chunks half, half + 2, ...
    const uint32_t stg0 = smem_u32(stg_base) + (uint32_t)((warp - 4) * (kStgTilesPerWarp * kStgTile));
    const uint32_t tempty_leader = smem_u32(&tempty_bar[0]) & 0xFEFFFFFFu;  // the pair leader's barrier (peer bit cleared); + 8 * stage
    if (MODE == ROUTE) {
      constexpr int KE = KMAX > 0 ? KMAX : 2;
      RouteSmem<KE>* rs = reinterpret_cast<RouteSmem<KE>*>(stg_base);
      {  // slot map and cleared histograms, visible to all epilogue warps before the first tile
        const int tid = threadIdx.x - 128;
        for (int i = tid; i < 128; i += kEpiWarps * 32) {
          const int sl = i < p.r.E ? p.r.slot_of[i] : -1;
          rs->slot[i] = sl;
          rs->zb[i] = (i >= p.r.E || (p.r.forced_local && sl < 0)) ? -INFINITY : (p.r.bias ? p.r.bias[i] : 0.f);
        }
        for (int i = tid; i < kAccStages * 128; i += kEpiWarps * 32) (&rs->hist[0][0])[i] = 0;
        bar_sync_named(5, kEpiWarps * 32);
      }
      int as = 0;
      uint32_t aphase = 0;
      for (long id = cluster_id; id < sched.total; id += n_clusters) {
        const Tile t = sched.decode(id);
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + as * BN;
        mbar_wait(smem_u32(&tfull_bar[as]), aphase);
        tc_fence_after();
        if constexpr (KMAX > kNetK) route_tile_epilogue<KMAX>(p, rs, taddr, q, half, lane, as, t.row0, t.live);
        else route_tile_epilogue_net<(KMAX > 0 ? KMAX : 2)>(p, rs, taddr, q, half, lane, as, t.row0, t.live);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(tempty_leader + 8 * as);
        if (++as == kAccStages) { as = 0; aphase ^= 1; }
      }
    } else if (MODE == DH) {
      // SwiGLU backward needs two saved factors (silu'(a) u and silu(a), "a" and "u" below) for every output element.
      // They are streamed global -> shared with cp.async,
      // kDhDepth 32-column chunks ahead of the consumer and across tile boundaries (the schedule is static), so the
      // loads never sit on the critical path of the accumulator drain.  A ring slot (a tile | u tile) is overwritten in
      // place with (da | du) and stored from there.
      long pid = cluster_id;                                  // prefetch cursor: (tile, chunk) in consumption order
      int pcc = half;
      bool pvalid = pid < sched.total;
      Tile pt = pvalid ? sched.decode(pid) : Tile{};
      const bf16* in_second = p.in1 ? p.in1 : p.in_h;
      auto issue = [&](int slot) {
        while (pvalid && pt.n_tile * BN + pcc * 32 >= p.F) {  // this warp has no (more) chunk in the tile
          pcc = half;
          pid += n_clusters;
          pvalid = pid < sched.total;
          if (pvalid) pt = sched.decode(pid);
        }
        if (pvalid) {
          const int prow0 = pt.row0 + q * 32;
          const int prows = !pt.live ? 0 : dense ? min(32, p.dense_rows - prow0) : 32;
          const size_t off = (size_t)prow0 * p.ld + (size_t)pt.part * p.F + pt.n_tile * BN + pcc * 32;
          const uint32_t sa = stg0 + slot * 2 * kStgTile, su = sa + kStgTile;
          if (prows > 0) {
#pragma unroll
            for (int it = 0; it < 4; ++it) {
              const int r = it * 8 + (lane >> 2), c = lane & 3;
              const bool ok = r < prows;
              const size_t g = off + (size_t)(ok ? r : 0) * p.ld + c * 8;
              cp_async16(sa + stg_off(r, c), p.in0 + g, ok);
              if (in_second) cp_async16(su + stg_off(r, c), in_second + g, ok);   // SwiGLU: silu(a); two-matrix expert: h (or nothing)
            }
          }
          pcc += 2;
          if (pcc >= BN / 32) {
            pcc = half;
            pid += n_clusters;
            pvalid = pid < sched.total;
            if (pvalid) pt = sched.decode(pid);
          }
        }
        cp_async_commit();
      };
#pragma unroll
      for (int sidx = 0; sidx < kDhDepth; ++sidx) issue(sidx);
      int slot = 0, as = 0;
      uint32_t aphase = 0;
      for (long id = cluster_id; id < sched.total; id += n_clusters) {
        const Tile t = sched.decode(id);
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + as * BN;
        const int row0 = t.row0 + q * 32;
        const int rows_valid = !t.live ? 0 : dense ? min(32, p.dense_rows - row0) : 32;
        const size_t base = (size_t)row0 * p.ld + (size_t)t.part * p.F;
        mbar_wait(smem_u32(&tfull_bar[as]), aphase);
        tc_fence_after();
        float dg_acc = 0.f;   // <dh, h> over this warp's chunks of the tile, for this lane's row
#pragma unroll 1
        for (int cc = half; cc < BN / 32; cc += 2) {
          const int n = t.n_tile * BN + cc * 32;
          if (n >= p.F) break;
          const uint32_t sa = stg0 + slot * 2 * kStgTile, su = sa + kStgTile;
          float dh[32];
          if (rows_valid > 0) tmem_ld32(taddr + cc * 32, dh);
          cp_async_wait<kDhDepth - 1>();
          __syncwarp();
          if (rows_valid > 0) {
            tmem_ld_wait();
#pragma unroll
            for (int g8 = 0; g8 < 4; ++g8) {
              const uint32_t o = stg_off(lane, g8);
              uint4 wa = lds128(sa + o), wu = in_second ? lds128(su + o) : make_uint4(0u, 0u, 0u, 0u);
              uint32_t* pa = reinterpret_cast<uint32_t*>(&wa);
              uint32_t* pu = reinterpret_cast<uint32_t*>(&wu);
#pragma unroll
              for (int i = 0; i < 4; ++i) {   // in0 = silu'(a) u, in1 = silu(a) (FWD1 epilogue): da = dh in0, du = dh in1
                const float2 a2 = unpack_bf16x2(pa[i]), u2 = unpack_bf16x2(pu[i]);
                const float d0 = dh[g8 * 8 + 2 * i], d1 = dh[g8 * 8 + 2 * i + 1];
                pa[i] = pack_bf16x2(d0 * a2.x, d1 * a2.y);
                if (p.in1) pu[i] = pack_bf16x2(d0 * u2.x, d1 * u2.y);
                else { dg_acc = fmaf(d0, u2.x, dg_acc); dg_acc = fmaf(d1, u2.y, dg_acc); }   // second stream = h: gate gradient
              }
              sts128(sa + o, wa);   // da over a, du over u: every lane rewrites exactly the bytes it read
              if (p.in1) sts128(su + o, wu);
            }
            __syncwarp();
            stg_to_global(sa, p.out0 + base + n, p.ld, lane, rows_valid);
            if (p.in1) stg_to_global(su, p.out1 + base + n, p.ld, lane, rows_valid);
          }
          __syncwarp();
          issue(slot);                                        // refill the slot just stored from
          if (++slot == kDhDepth) slot = 0;
        }
        if (p.dgate_part && rows_valid > 0 && lane < rows_valid)
          p.dgate_part[(size_t)(row0 + lane) * p.n_dgate_parts + 2 * t.n_tile + half] = dg_acc;
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(tempty_leader + 8 * as);
        if (++as == kAccStages) { as = 0; aphase ^= 1; }
      }
      cp_async_wait<0>();
    } else {
    const uint32_t stg1 = stg0 + kStgTile, stg2 = stg1 + kStgTile;  // FWD1 only
    int st_buf = 0;                                                   // FWD2 / DX bulk stores: staging tile in turn
    int as = 0;
    uint32_t aphase = 0;
    for (long id = cluster_id; id < sched.total; id += n_clusters) {
      const Tile t = sched.decode(id);
      const bool have_acc = t.num_kb > 0;
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + as * BN;
      const int row0 = t.row0 + q * 32;   // first row (or WGRAD output row m) of this warp
      if (have_acc) { mbar_wait(smem_u32(&tfull_bar[as]), aphase); tc_fence_after(); }
      if (MODE == WGRAD) {
        const int rows_valid = !t.live ? 0 : min(32, t.M - row0);
        bf16* obase = (p.n_jobs > 0 ? p.job_out[t.job] : p.out0) + ((size_t)t.group * t.M + row0) * t.N;
#pragma unroll 1
        for (int cc = half; cc < BN / 32 && rows_valid > 0; cc += 2) {
          const int n = t.n_tile * BN + cc * 32;
          if (n >= t.N) break;
          float v[32];
          if (have_acc) { tmem_ld32(taddr + cc * 32, v); tmem_ld_wait(); }
          else {
#pragma unroll
            for (int i = 0; i < 32; ++i) v[i] = 0.f;
          }
          if (t.piece >= 0) {  // K piece of a tail tile: fp32, tile-local layout [piece][cta][128][256]
            if (lane < rows_valid) {
              float4* dst = reinterpret_cast<float4*>(p.tail_part + (((size_t)t.piece * 2 + rank) * BM + q * 32 + lane) * BN + cc * 32);
#pragma unroll
              for (int i = 0; i < 8; ++i) dst[i] = make_float4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
            }
            continue;
          }
          if (p.out_f32) {  // split-K partials (small): one 128-byte row segment per thread
            if (lane < rows_valid) {
              float4* dst = reinterpret_cast<float4*>(p.out_f32 + ((size_t)t.group * p.M + row0 + lane) * p.N + n);
#pragma unroll
              for (int i = 0; i < 8; ++i) dst[i] = make_float4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
            }
            continue;
          }
          stg_put_row(stg0, lane, v);
          __syncwarp();
          stg_to_global(stg0, obase + n, t.N, lane, rows_valid);
          __syncwarp();
        }
      } else {
        const int rows_valid = !t.live ? 0 : dense ? min(32, p.dense_rows - row0) : 32;
        if (MODE == FWD1) {
          const size_t base = (size_t)row0 * p.ld + (size_t)t.part * p.F;
#pragma unroll 1
          for (int cc = half; cc < (BN / 2) / 32 && rows_valid > 0; cc += 2) {
            const int n = t.n_tile * (BN / 2) + cc * 32;
            if (n >= p.F) break;
            float a[32], u[32], sa_h[32];
            tmem_ld32(taddr + cc * 32, a);
            tmem_ld32(taddr + BN / 2 + cc * 32, u);
            tmem_ld_wait();
            // what the backward needs of (a, u) is only silu(a) and d silu(a)/da * u: save those (same bytes as a, u), so
            // the DH epilogue is two multiplies per element instead of a sigmoid (it is epilogue-bound at small d)
#pragma unroll
            for (int i = 0; i < 32; ++i) {
              const float sg = __fdividef(1.0f, 1.0f + __expf(-a[i]));
              const float sa = a[i] * sg;                                   // silu(a)
              a[i] = fmaf(sa, 1.0f - sg, sg) * u[i];                         // silu'(a) * u = s (1 + a (1 - s)) u
              const float h = sa * u[i];
              u[i] = sa;
              sa_h[i] = h;
            }
            if (p.tma_store) {   // three bulk tensor stores per chunk (maps m[3..5] = the outputs); the previous chunk's have been
              if (lane == 0) bulk_wait_read<0>();   // reading the tiles while this chunk's sigmoids were computed
              __syncwarp();
              stg_put_row_sw64(stg0, lane, a);
              stg_put_row_sw64(stg1, lane, u);
              stg_put_row_sw64(stg2, lane, sa_h);
              asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
              __syncwarp();
              if (lane == 0) {
                const int c0 = t.part * p.F + n;
                tma_store_2d(&maps.m[3], stg0, c0, row0);
                tma_store_2d(&maps.m[4], stg1, c0, row0);
                tma_store_2d(&maps.m[5], stg2, c0, row0);
                bulk_commit();
              }
              continue;
            }
            stg_put_row(stg0, lane, a);
            stg_put_row(stg1, lane, u);
            stg_put_row(stg2, lane, sa_h);
            __syncwarp();
            stg_to_global(stg0, p.out0 + base + n, p.ld, lane, rows_valid);
            stg_to_global(stg1, p.out1 + base + n, p.ld, lane, rows_valid);
            stg_to_global(stg2, p.out2 + base + n, p.ld, lane, rows_valid);
            __syncwarp();
          }
        } else if (MODE == FWD1S) {   // two-matrix expert: h = silu(a); out0 <- silu'(a) (the backward's factor), out2 <- h
          const size_t base = (size_t)row0 * p.ld + (size_t)t.part * p.F;
#pragma unroll 1
          for (int cc = half; cc < BN / 32 && rows_valid > 0; cc += 2) {
            const int n = t.n_tile * BN + cc * 32;
            if (n >= p.F) break;
            float a[32], h[32];
            tmem_ld32(taddr + cc * 32, a);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) {
              const float sg = __fdividef(1.0f, 1.0f + __expf(-a[i]));
              h[i] = a[i] * sg;                          // silu(a)
              a[i] = fmaf(h[i], 1.0f - sg, sg);           // silu'(a) = s (1 + a (1 - s))
            }
            if (p.tma_store) {   // (maps m[3], m[5] = out0, out2)
              if (lane == 0) bulk_wait_read<0>();
              __syncwarp();
              stg_put_row_sw64(stg0, lane, a);
              stg_put_row_sw64(stg1, lane, h);
              asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
              __syncwarp();
              if (lane == 0) {
                const int c0 = t.part * p.F + n;
                tma_store_2d(&maps.m[3], stg0, c0, row0);
                tma_store_2d(&maps.m[5], stg1, c0, row0);
                bulk_commit();
              }
              continue;
            }
            stg_put_row(stg0, lane, a);
            stg_put_row(stg1, lane, h);
            __syncwarp();
            stg_to_global(stg0, p.out0 + base + n, p.ld, lane, rows_valid);
            stg_to_global(stg1, p.out2 + base + n, p.ld, lane, rows_valid);
            __syncwarp();
          }
        } else if (p.tma_store) {  // FWD2, DX: [rows, d] tile, one bulk tensor store per 32 x 32 chunk (rows beyond the tensor are clipped)
#pragma unroll 1
          for (int cc = half; cc < BN / 32 && rows_valid > 0; cc += 2) {
            const int n = t.n_tile * BN + cc * 32;
            if (n >= p.d) break;
            float v[32];
            tmem_ld32(taddr + cc * 32, v);
            tmem_ld_wait();
            const uint32_t stg = stg0 + st_buf * kStgTile;
            if (lane == 0) bulk_wait_read<1>();       // the store that last read this tile (two chunks ago) has its data
            __syncwarp();
            stg_put_row_sw64(stg, lane, v);
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> the bulk store's async-proxy reads
            __syncwarp();
            if (lane == 0) { tma_store_2d(&maps.m[4], stg, n, row0); bulk_commit(); }
            st_buf ^= 1;
          }
        } else {  // FWD2, DX: plain store of a [rows, d] tile
#pragma unroll 1
          for (int cc = half; cc < BN / 32 && rows_valid > 0; cc += 2) {
            const int n = t.n_tile * BN + cc * 32;
            if (n >= p.d) break;
            float v[32];
            tmem_ld32(taddr + cc * 32, v);
            tmem_ld_wait();
            stg_put_row(stg0, lane, v);
            __syncwarp();
            stg_to_global(stg0, p.out0 + (size_t)row0 * p.d + n, p.d, lane, rows_valid);
            __syncwarp();
          }
        }
      }
      if (have_acc) {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(tempty_leader + 8 * as);
        if (++as == kAccStages) { as = 0; aphase ^= 1; }
      }
    }
    if ((MODE == FWD2 || MODE == DX || MODE == FWD1 || MODE == FWD1S) && p.tma_store && lane == 0) bulk_wait_all();   // shared memory stays valid until the stores have read it
    }
  }

  // neither CTA may leave (or free tensor memory) while its peer can still read its shared memory or signal its barriers
  tc_fence_before();
  cluster_sync_all();
  if (warp == 2) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols) : "memory");
  }
}

// Adds the K pieces of the tail tiles (fixed order) and writes them as bf16 into dW.  grid = (tail tiles, 2 CTAs of a pair, 8 row slabs).
__global__ void __launch_bounds__(256)
wgrad_tail_fixup_kernel(const float* __restrict__ part, int tail_first, int ks, int m_pairs, int n_tiles_n, int M, int N,
                        bf16* __restrict__ out) {
  pdl_launch_dependents();
  pdl_wait();
  const int u = blockIdx.x, rank = blockIdx.y;
  const long tile = (long)tail_first + u;
  const int group = (int)(tile / ((long)m_pairs * n_tiles_n)), rem = (int)(tile % ((long)m_pairs * n_tiles_n));
  const int row0 = (rem / n_tiles_n) * 2 * BM + rank * BM, n0 = (rem % n_tiles_n) * BN;
  // blockIdx.z: 16-row slab of the CTA's 128 rows
  for (int e = blockIdx.z * 16 * BN + threadIdx.x * 4; e < (blockIdx.z + 1) * 16 * BN; e += 256 * 4) {
    const int r = e / BN, cidx = e % BN;
    if (row0 + r >= M || n0 + cidx >= N) continue;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int j = 0; j < ks; ++j) {
      const float4 v = *reinterpret_cast<const float4*>(part + (((size_t)(u * ks + j) * 2 + rank) * BM + r) * BN + cidx);
      acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    uint2 o;
    o.x = pack_bf16x2(acc.x, acc.y);
    o.y = pack_bf16x2(acc.z, acc.w);
    *reinterpret_cast<uint2*>(out + ((size_t)group * M + row0 + r) * N + n0 + cidx) = o;
  }
}

// ---------------------------------------------------------------------------------------------------------
// host side: tensor maps and launches
// ---------------------------------------------------------------------------------------------------------
template <int MODE, int KMAX = 0>
int launch(const TmaMaps& maps, const UmmaParams& p, cudaStream_t st, const char* name) {
  static PerDeviceOnce attr;
  if (attr.need()) {
    FOMOE_CUDA_OK(cudaFuncSetAttribute(umma_grouped_kernel<MODE, KMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes_of(MODE, KMAX)));
    attr.set();
  }
  FOMOE_CUDA_OK(launch_pdl(umma_grouped_kernel<MODE, KMAX>, num_sms() & ~1, kThreads, smem_bytes_of(MODE, KMAX), st, maps, p));
  FOMOE_LAUNCH_OK(name);
  return FOMOE_OK;
}

}  // namespace

// FWD2 / DX output through TMA bulk stores: m[4] = [rows, d] with a {32 columns, 32 rows} box, 64-byte swizzle.  FOMOE_TMA_STORE=0
// in the environment keeps the st.global epilogue (A/B measurements).
static bool tma_store_enabled() {
  static const bool on = [] { const char* e = getenv("FOMOE_TMA_STORE"); return !(e && e[0] == '0'); }();
  return on;
}
static bool set_store_map(TmaMaps& m, UmmaParams& q, const void* out, uint64_t rows, int d) {
  q.tma_store = 0;
  if (!tma_store_enabled()) return true;
  if (!make_map_box(&m.m[4], out, (uint64_t)d, rows, (uint64_t)d, 32, 32, CU_TENSOR_MAP_SWIZZLE_64B)) return false;
  q.tma_store = 1;
  return true;
}

// FWD1 / FWD1S: m[3], m[4], m[5] = out0, out1, out2 ([rows, ld]); a NULL output is skipped
static bool set_store_maps3(TmaMaps& m, UmmaParams& q, uint64_t rows, int ld) {
  q.tma_store = 0;
  if (!tma_store_enabled()) return true;
  const void* outs[3] = {q.out0, q.out1, q.out2};
  for (int i = 0; i < 3; ++i)
    if (outs[i] && !make_map_box(&m.m[3 + i], outs[i], (uint64_t)ld, rows, (uint64_t)ld, 32, 32, CU_TENSOR_MAP_SWIZZLE_64B)) return false;
  q.tma_store = 1;
  return true;
}

bool umma_supported(const fomoe_config& c) {
  if (c.dtype != FOMOE_BF16) return false;
  if (c.d_model % 64 || c.d_ff % 64) return false;
  if (c.n_shared > 0 && c.d_ff_shared % 64) return false;
  return true;
}

// Router logits + gate + top-k + mask + per-block histogram (ROUTE mode).  wr_split: [d, NP] bf16 pieces of W_r, NP = 128 or 256.
int umma_route(const fomoe_config& c, const void* x, const void* wr_split, int NP, int Epad, int pieces, const float* bias, int n_res,
               const fomoe_route_state& out, const RouteWs& ws, cudaStream_t st) {
  UmmaParams p{};
  p.dense_rows = c.T; p.parts = 1; p.d = c.d_model; p.F = NP; p.ld = NP; p.N = NP;
  p.r = RouteEpi{c.E, Epad, pieces, c.top_k, c.gate_fn, c.gate_rule, n_res, c.route_mode == FOMOE_ROUTE_FORCED_LOCAL ? 1 : 0,
                 1.0f / c.temperature, bias, ws.slot_of,
                 out.probs, out.topk_idx, out.gate, ws.blk_hist};
  TmaMaps m{};
  MAP_OK(make_map(&m.m[0], x, c.d_model, c.T, c.d_model, 128));
  MAP_OK(make_map(&m.m[1], wr_split, NP, c.d_model, NP, 64));
  m.m[2] = m.m[3] = m.m[0];
  if (c.top_k <= 2) return launch<ROUTE, 2>(m, p, st, "umma_grouped_kernel<ROUTE>");
  if (c.top_k <= 4) return launch<ROUTE, 4>(m, p, st, "umma_grouped_kernel<ROUTE>");
  if (c.top_k <= 8) return launch<ROUTE, 8>(m, p, st, "umma_grouped_kernel<ROUTE>");
  if (c.top_k <= 16) return launch<ROUTE, 16>(m, p, st, "umma_grouped_kernel<ROUTE>");   // Table 1: N_active up to 32
  return launch<ROUTE, 32>(m, p, st, "umma_grouped_kernel<ROUTE>");
}

int umma_ffn_fwd(const fomoe_config& c, int n_res, const void* x, const RouteWs& rws, const ActWs& aws, const ScratchWs& sws,
                 const FfnPtrs& w, cudaStream_t st) {
  const int d = c.d_model, F = c.d_ff;
  const bool silu = c.expert_fn == FOMOE_EXPERT_SILU;
  if (n_res > 0 && c.T > 0) {
    const uint64_t R = (uint64_t)rws.R_cap;
    UmmaParams p{};
    p.n_mtiles = rws.n_mtiles; p.tile_slot = rws.tile_slot; p.pair_info = rws.pair_info; p.parts = 1; p.d = d; p.F = F; p.ld = F;
    if (silu && (fine_mask(c) & 1)) {   // d_expert = 128: x rows gathered inside the kernel (fine_gemm.cu)
      int rc = fine_fwd1(c, n_res, x, rws, aws, w.w_up, st);
      if (rc != FOMOE_OK) return rc;
    } else if (silu) {   // two-matrix expert: a = X W_up^T, h = silu(a)
      TmaMaps m{};
      MAP_OK(make_map(&m.m[0], aws.xp, d, R, d, 128));
      MAP_OK(make_map(&m.m[1], w.w_up, d, (uint64_t)n_res * F, d, 128));
      m.m[2] = m.m[3] = m.m[0];
      UmmaParams q = p;
      q.out0 = (bf16*)aws.a; q.out2 = (bf16*)aws.h;
      MAP_OK(set_store_maps3(m, q, R, F));
      int rc = launch<FWD1S>(m, q, st, "umma_grouped_kernel<FWD1S>");
      if (rc != FOMOE_OK) return rc;
    } else {
      TmaMaps m{};
      MAP_OK(make_map(&m.m[0], aws.xp, d, R, d, 128));
      MAP_OK(make_map(&m.m[1], w.w_gate, d, (uint64_t)n_res * F, d, 128));
      MAP_OK(make_map(&m.m[2], w.w_up, d, (uint64_t)n_res * F, d, 128));
      m.m[3] = m.m[0];
      UmmaParams q = p;
      q.out0 = (bf16*)aws.a; q.out1 = (bf16*)aws.u; q.out2 = (bf16*)aws.h;
      MAP_OK(set_store_maps3(m, q, R, F));
      int rc = launch<FWD1>(m, q, st, "umma_grouped_kernel<FWD1>");
      if (rc != FOMOE_OK) return rc;
    }
    {
      TmaMaps m{};
      MAP_OK(make_map(&m.m[0], aws.h, F, R, F, 128));
      MAP_OK(make_map(&m.m[1], w.w_down, F, (uint64_t)n_res * d, F, 128));
      m.m[2] = m.m[3] = m.m[0];
      UmmaParams q = p;
      q.out0 = (bf16*)aws.o;
      MAP_OK(set_store_map(m, q, aws.o, R, d));
      int rc = launch<FWD2>(m, q, st, "umma_grouped_kernel<FWD2>");
      if (rc != FOMOE_OK) return rc;
    }
  }
  if (c.n_shared > 0 && c.T > 0) {
    const int Fs = c.d_ff_shared, ns = c.n_shared, ld = ns * Fs;
    UmmaParams p{};
    p.dense_rows = c.T; p.parts = ns; p.d = d; p.F = Fs; p.ld = ld;
    if (silu) {
      TmaMaps m{};
      MAP_OK(make_map(&m.m[0], x, d, c.T, d, 128));
      MAP_OK(make_map(&m.m[1], w.sh_up, d, (uint64_t)ns * Fs, d, 128));
      m.m[2] = m.m[3] = m.m[0];
      UmmaParams q = p;
      q.out0 = (bf16*)aws.sa; q.out2 = (bf16*)aws.sh;
      MAP_OK(set_store_maps3(m, q, c.T, ld));
      int rc = launch<FWD1S>(m, q, st, "umma_grouped_kernel<FWD1S,shared>");
      if (rc != FOMOE_OK) return rc;
    } else {
      TmaMaps m{};
      MAP_OK(make_map(&m.m[0], x, d, c.T, d, 128));
      MAP_OK(make_map(&m.m[1], w.sh_gate, d, (uint64_t)ns * Fs, d, 128));
      MAP_OK(make_map(&m.m[2], w.sh_up, d, (uint64_t)ns * Fs, d, 128));
      m.m[3] = m.m[0];
      UmmaParams q = p;
      q.out0 = (bf16*)aws.sa; q.out1 = (bf16*)aws.su; q.out2 = (bf16*)aws.sh;
      MAP_OK(set_store_maps3(m, q, c.T, ld));
      int rc = launch<FWD1>(m, q, st, "umma_grouped_kernel<FWD1,shared>");
      if (rc != FOMOE_OK) return rc;
    }
    {
      TmaMaps m{};
      MAP_OK(make_map(&m.m[0], aws.sh, ld, c.T, ld, 128));
      MAP_OK(make_map(&m.m[1], w.sh_down, Fs, (uint64_t)ns * d, Fs, 128));
      m.m[2] = m.m[3] = m.m[0];
      UmmaParams q = p;
      q.out0 = (bf16*)sws.y_sh;
      MAP_OK(set_store_map(m, q, sws.y_sh, c.T, d));
      int rc = launch<FWD2>(m, q, st, "umma_grouped_kernel<FWD2,shared>");
      if (rc != FOMOE_OK) return rc;
    }
  }
  return FOMOE_OK;
}

int umma_ffn_bwd(const fomoe_config& c, int n_res, const void* x, const void* dy, const RouteWs& rws, const ActWs& aws,
                 const ScratchWs& sws, const FfnPtrs& w, void* dw_gate, void* dw_up, void* dw_down, void* d_sh_gate,
                 void* d_sh_up, void* d_sh_down, cudaStream_t st_main, bool dgate_in_dh, const std::function<int()>* after_dh,
                 cudaStream_t wg_stream, cudaEvent_t wg_fork, bool* wg_forked) {
  const int d = c.d_model, F = c.d_ff;
  const bool silu = c.expert_fn == FOMOE_EXPERT_SILU;   // two-matrix expert: one saved factor, dxp = dA W_up, dW_up = dA^T x
  // Two phases over the same code: 0 = every data gradient (DH, DX; routed, then shared), 1 = every weight gradient.  The
  // weight gradients depend on the DH outputs only, the dx scatter-sum (the caller's next launch) on the DX outputs only: with
  // a second stream the bandwidth-bound scatter-sum runs beside the weight-gradient GEMMs instead of after them.
  auto phase_fn = [&](const int phase, cudaStream_t st) -> int {
  if (n_res > 0) {
    const uint64_t R = (uint64_t)rws.R_cap;
    UmmaParams p{};
    p.n_mtiles = rws.n_mtiles; p.tile_slot = rws.tile_slot; p.pair_info = rws.pair_info; p.pad_offsets = rws.pad_offsets; p.pad_end64 = rws.pad_end64; p.parts = 1; p.d = d; p.F = F; p.ld = F;
    const int fine = silu ? fine_mask(c) : 0;
    void* hg = sws.du;    // fine path: g h [R, F] (the two-matrix expert has no du)
    if (c.T > 0 && phase == 0) {
      if (fine & 2) {  // dh = dy[token] W_down gathered in the kernel; da, hg = g h and <dh, h> out of its epilogue
        int rc = fine_dh(c, n_res, dy, rws, aws, sws, hg, w.w_down, st);
        if (rc != FOMOE_OK) return rc;
        if (after_dh) { rc = (*after_dh)(); if (rc != FOMOE_OK) return rc; }
      } else {  // dh = dO W_down, fused SwiGLU backward
        TmaMaps m{};
        MAP_OK(make_map(&m.m[0], sws.dop, d, R, d, 128));
        MAP_OK(make_map(&m.m[1], w.w_down, F, (uint64_t)n_res * d, F, 64));
        m.m[2] = m.m[3] = m.m[0];
        UmmaParams q = p;
        q.in0 = (const bf16*)aws.a; q.in1 = silu ? nullptr : (const bf16*)aws.u; q.out0 = (bf16*)sws.da; q.out1 = (bf16*)sws.du;
        if (dgate_in_dh && silu) { q.in_h = (const bf16*)aws.h; q.dgate_part = sws.dgate_part; q.n_dgate_parts = sws.n_dgate_parts; }
        int rc = launch<DH>(m, q, st, "umma_grouped_kernel<DH>");
        if (rc != FOMOE_OK) return rc;
        if (after_dh) { rc = (*after_dh)(); if (rc != FOMOE_OK) return rc; }
      }
      {  // dxp = dA W_gate + dU W_up
        TmaMaps m{};
        MAP_OK(make_map(&m.m[0], sws.da, F, R, F, 128));
        MAP_OK(make_map(&m.m[1], silu ? sws.da : sws.du, F, R, F, 128));
        MAP_OK(make_map(&m.m[2], silu ? w.w_up : w.w_gate, d, (uint64_t)n_res * F, d, 64));
        MAP_OK(make_map(&m.m[3], w.w_up, d, (uint64_t)n_res * F, d, 64));
        UmmaParams q = p;
        q.ksegs = silu ? 1 : 2;
        q.out0 = (bf16*)sws.dxp;
        MAP_OK(set_store_map(m, q, sws.dxp, R, d));
        int rc = launch<DX>(m, q, st, "umma_grouped_kernel<DX>");
        if (rc != FOMOE_OK) return rc;
      }
    }
    // weight gradients, K = the slot's padded rows (padding rows are zero)
    struct WG { const void* A; int lda; const void* B; int ldb; int M, N; void* out; };
    const WG jobs[3] = {{sws.dop, d, aws.h, F, d, F, dw_down}, {sws.da, F, aws.xp, d, F, d, silu ? dw_up : dw_gate},
                        {sws.du, F, aws.xp, d, F, d, dw_up}};
    if (phase == 0) {
    } else if (fine & 4) {
      int rc = fine_wgrad(c, n_res, x, dy, rws, sws, hg, dw_up, dw_down, st);
      if (rc != FOMOE_OK) return rc;
    } else {   // one launch for all of them (same row groups, same K ranges)
      TmaMaps m{};
      UmmaParams q = p;
      const int nj = silu ? 2 : 3;
      for (int ji = 0; ji < nj; ++ji) {
        const WG& j = jobs[ji];
        MAP_OK(make_map(&m.m[2 * ji], j.A, j.lda, R, j.lda, 64));
        MAP_OK(make_map(&m.m[2 * ji + 1], j.B, j.ldb, R, j.ldb, 64));
        q.job_M[ji] = j.M; q.job_N[ji] = j.N; q.job_out[ji] = (bf16*)j.out; q.job_agcol[ji] = 0; q.job_bgcol[ji] = 0;
      }
      for (int i = 2 * nj; i < 6; ++i) m.m[i] = m.m[0];
      q.n_jobs = nj; q.n_groups = n_res; q.M = jobs[0].M; q.N = jobs[0].N; q.a_gcol = 0; q.b_gcol = 0; q.out0 = (bf16*)jobs[0].out;
      int rc = launch<WGRAD>(m, q, st, "umma_grouped_kernel<WGRAD>");
      if (rc != FOMOE_OK) return rc;
    }
  }
  if (c.n_shared > 0 && c.T == 0) {  // empty batch: exact zeros
    if (phase == 0) return FOMOE_OK;
    const size_t n = sizeof(bf16) * (size_t)c.n_shared * c.d_ff_shared * d;
    if (!silu) FOMOE_CUDA_OK(cudaMemsetAsync(d_sh_gate, 0, n, st));
    FOMOE_CUDA_OK(cudaMemsetAsync(d_sh_up, 0, n, st));
    FOMOE_CUDA_OK(cudaMemsetAsync(d_sh_down, 0, n, st));
  } else if (c.n_shared > 0) {
    const int Fs = c.d_ff_shared, ns = c.n_shared, ld = ns * Fs;
    UmmaParams p{};
    p.dense_rows = c.T; p.parts = ns; p.d = d; p.F = Fs; p.ld = ld;
    if (c.T > 0 && phase == 0) {
      {
        TmaMaps m{};
        MAP_OK(make_map(&m.m[0], dy, d, c.T, d, 128));
        MAP_OK(make_map(&m.m[1], w.sh_down, Fs, (uint64_t)ns * d, Fs, 64));
        m.m[2] = m.m[3] = m.m[0];
        UmmaParams q = p;
        q.in0 = (const bf16*)aws.sa; q.in1 = silu ? nullptr : (const bf16*)aws.su; q.out0 = (bf16*)sws.dsa; q.out1 = (bf16*)sws.dsu;
        int rc = launch<DH>(m, q, st, "umma_grouped_kernel<DH,shared>");
        if (rc != FOMOE_OK) return rc;
      }
      {
        TmaMaps m{};
        MAP_OK(make_map(&m.m[0], sws.dsa, ld, c.T, ld, 128));
        MAP_OK(make_map(&m.m[1], silu ? sws.dsa : sws.dsu, ld, c.T, ld, 128));
        MAP_OK(make_map(&m.m[2], silu ? w.sh_up : w.sh_gate, d, (uint64_t)ns * Fs, d, 64));
        MAP_OK(make_map(&m.m[3], w.sh_up, d, (uint64_t)ns * Fs, d, 64));
        UmmaParams q = p;
        q.ksegs = silu ? 1 : 2;
        q.out0 = (bf16*)sws.dx_sh;
        MAP_OK(set_store_map(m, q, sws.dx_sh, c.T, d));
        int rc = launch<DX>(m, q, st, "umma_grouped_kernel<DX,shared>");
        if (rc != FOMOE_OK) return rc;
      }
    }
    if (phase == 0) return FOMOE_OK;
    struct WG { const void* A; int lda; int a_gcol; const void* B; int ldb; int b_gcol; int M, N; void* out; };
    const WG jobs[3] = {{dy, d, 0, aws.sh, ld, Fs, d, Fs, d_sh_down},
                        {sws.dsa, ld, Fs, x, d, 0, Fs, d, silu ? d_sh_up : d_sh_gate},
                        {sws.dsu, ld, Fs, x, d, 0, Fs, d, d_sh_up}};
    // All weight gradients in ONE launch when their tiles together fill the scheduler rounds (C3: 3 x 96 tiles = 3.9 rounds of
    // 74 pairs); otherwise one launch each, with the last round cut into K pieces.
    const int nj = silu ? 2 : 3, pairs_all = (num_sms() & ~1) / 2;
    long tiles_all = 0;
    for (int ji = 0; ji < nj; ++ji) tiles_all += (long)ns * ceil_div(jobs[ji].M, 2 * BM) * ceil_div(jobs[ji].N, BN);
    const bool merged = (double)tiles_all / (double)(((tiles_all + pairs_all - 1) / pairs_all) * pairs_all) >= 0.85;
    if (merged) {
      TmaMaps m{};
      UmmaParams q = p;
      for (int ji = 0; ji < nj; ++ji) {
        const WG& j = jobs[ji];
        MAP_OK(make_map(&m.m[2 * ji], j.A, j.lda, c.T, j.lda, 64));
        MAP_OK(make_map(&m.m[2 * ji + 1], j.B, j.ldb, c.T, j.ldb, 64));
        q.job_M[ji] = j.M; q.job_N[ji] = j.N; q.job_out[ji] = (bf16*)j.out; q.job_agcol[ji] = j.a_gcol; q.job_bgcol[ji] = j.b_gcol;
      }
      for (int i = 2 * nj; i < 6; ++i) m.m[i] = m.m[0];
      q.n_jobs = nj; q.n_groups = ns; q.M = jobs[0].M; q.N = jobs[0].N; q.out0 = (bf16*)jobs[0].out;
      int rc = launch<WGRAD>(m, q, st, "umma_grouped_kernel<WGRAD,shared>");
      if (rc != FOMOE_OK) return rc;
    }
    for (int ji = 0; ji < (merged ? 0 : nj); ++ji) {
      const WG& j = jobs[ji];
      TmaMaps m{};
      MAP_OK(make_map(&m.m[0], j.A, j.lda, c.T, j.lda, 64));
      MAP_OK(make_map(&m.m[1], j.B, j.ldb, c.T, j.ldb, 64));
      m.m[2] = m.m[3] = m.m[0];
      UmmaParams q = p;
      q.n_groups = ns; q.M = j.M; q.N = j.N; q.a_gcol = j.a_gcol; q.b_gcol = j.b_gcol; q.out0 = (bf16*)j.out;
      // few long tiles (K = T): cut the tiles of the last, partially filled round into K pieces so that it fills the pairs
      const int m_pairs = ceil_div(j.M, 2 * BM), ntn = ceil_div(j.N, BN), tiles = ns * m_pairs * ntn, pairs = (num_sms() & ~1) / 2;
      const int tail = tiles % pairs;
      int ks = tail > 0 ? pairs / tail : 1;
      if (ks > kTailSplitMax) ks = kTailSplitMax;
      while (ks > 1 && c.T / ks < 2048) --ks;
      if (ks > 1 && j.N % 4 == 0) {
        q.tail_first = tiles - tail; q.tail_ks = ks; q.tail_chunk = ceil_div(ceil_div(c.T, ks), BK) * BK; q.tail_part = sws.wg_tail;
      } else {
        ks = 1;
      }
      int rc = launch<WGRAD>(m, q, st, "umma_grouped_kernel<WGRAD,shared>");
      if (rc != FOMOE_OK) return rc;
      if (ks > 1) {
        FOMOE_CUDA_OK(launch_pdl(wgrad_tail_fixup_kernel, dim3(tail, 2, 8), 256, 0, st, (const float*)sws.wg_tail, tiles - tail, ks, m_pairs, ntn,
                                 j.M, j.N, (bf16*)j.out));
        FOMOE_LAUNCH_OK("wgrad_tail_fixup_kernel");
      }
    }
  }
  return FOMOE_OK;
  };   // phase_fn
  int rc = phase_fn(0, st_main);
  if (rc != FOMOE_OK) return rc;
  cudaStream_t wst = st_main;
  if (wg_stream && wg_fork) {   // the weight gradients wait for everything queued on the main stream so far (DH and DX)
    FOMOE_CUDA_OK(cudaEventRecord(wg_fork, st_main));
    FOMOE_CUDA_OK(cudaStreamWaitEvent(wg_stream, wg_fork, 0));
    if (wg_forked) *wg_forked = true;
    wst = wg_stream;
  }
  return phase_fn(1, wst);
}


namespace {
__global__ void wr_to_bf16_kernel(const float* __restrict__ w_r, int d, int E, int Ez, bf16* __restrict__ out) {
  pdl_launch_dependents();
  pdl_wait();
  const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long)d * Ez) return;
  const int i = (int)(idx / Ez), e = (int)(idx % Ez);
  out[idx] = __float2bfloat16_rn(e < E ? w_r[(size_t)i * E + e] : 0.f);
}
__global__ void reduce_wr_parts_kernel(const float* __restrict__ part, int n_parts, int d, int E, int Ez, float* __restrict__ out) {
  pdl_launch_dependents();
  pdl_wait();
  const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long)d * E) return;
  const int i = (int)(idx / E), e = (int)(idx % E);
  float s = 0.f;
  for (int g = 0; g < n_parts; ++g) s += part[((size_t)g * d + i) * Ez + e];  // fixed order
  out[idx] = s;
}
}  // namespace

int umma_router_bwd(const fomoe_config& c, const void* x, const float* w_router, const void* wr_bf, const ScratchWs& sws,
                    float* dw_router, cudaStream_t st) {
  const int d = c.d_model, E = c.E, Ez = sws.Ez, T = c.T;
  if (!wr_bf) {
    wr_bf = sws.wr_bf;
    const long n = (long)d * Ez;
    FOMOE_CUDA_OK(launch_pdl(wr_to_bf16_kernel, (unsigned)((n + 255) / 256), 256, 0, st, w_router, d, E, Ez, (bf16*)sws.wr_bf));
    FOMOE_LAUNCH_OK("wr_to_bf16_kernel");
  }
  {  // dx_r [T,d] = dz [T,Ez] W_r^T : FWD2 shape on dense rows (A = dz, K = Ez; B = W_r [d,Ez] K-major)
    UmmaParams p{};
    p.dense_rows = T; p.parts = 1; p.d = d; p.F = Ez; p.ld = Ez;
    TmaMaps m{};
    MAP_OK(make_map(&m.m[0], sws.dz_bf, Ez, T, Ez, 128));
    MAP_OK(make_map(&m.m[1], wr_bf, Ez, d, Ez, 128));
    m.m[2] = m.m[3] = m.m[0];
    p.out0 = (bf16*)sws.dx_r;
    MAP_OK(set_store_map(m, p, sws.dx_r, T, d));
    int rc = launch<FWD2>(m, p, st, "umma_grouped_kernel<FWD2,router dx>");
    if (rc != FOMOE_OK) return rc;
  }
  // dW_r [d,E] = x^T dz : WGRAD shape, split over tokens into G groups, fp32 partials, fixed-order reduce
  const int m_tiles = (d + BM - 1) / BM;
  int G = (2 * num_sms() + m_tiles - 1) / m_tiles;
  if (G > kRouterSplit) G = kRouterSplit;
  if (G > (T + 511) / 512) G = (T + 511) / 512;
  if (G < 1) G = 1;
  const int k_chunk = ((T + G - 1) / G + 63) / 64 * 64;
  G = (T + k_chunk - 1) / k_chunk;
  {
    UmmaParams p{};
    p.dense_rows = T; p.parts = 1; p.d = d; p.F = Ez; p.ld = Ez;
    p.n_groups = G; p.M = d; p.N = Ez; p.k_chunk = k_chunk; p.out_f32 = sws.dwr_part;
    TmaMaps m{};
    MAP_OK(make_map(&m.m[0], x, d, T, d, 64));
    MAP_OK(make_map(&m.m[1], sws.dz_bf, Ez, T, Ez, 64));
    m.m[2] = m.m[3] = m.m[0];
    int rc = launch<WGRAD>(m, p, st, "umma_grouped_kernel<WGRAD,router dW>");
    if (rc != FOMOE_OK) return rc;
  }
  {
    const long n = (long)d * E;
    FOMOE_CUDA_OK(launch_pdl(reduce_wr_parts_kernel, (unsigned)((n + 255) / 256), 256, 0, st, sws.dwr_part, G, d, E, Ez, dw_router));
    FOMOE_LAUNCH_OK("reduce_wr_parts_kernel");
  }
  return FOMOE_OK;
}

}  // namespace fomoe
