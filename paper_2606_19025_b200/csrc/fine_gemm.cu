// Fine-grained experts (the paper's own shapes: d_expert = 128, 4-32 active): the expert GEMMs with their
// token-indexed operand GATHERED inside the kernel, so that no permuted copy of x or of dy is ever written.
//
// With F = d_expert = 128 every GEMM of the step is a memory stream (one [P, d] operand against a 128-wide one), and the
// permuted copies xp = x[token(r)] and dop = g_r dy[token(r)] cost a write and 2-3 reads of [P, d] each.  The kernels here
// read those rows straight from x / dy (L2-resident: [T, d] is 16-64 MB) by token id:
//   F1  a = x[tok] W_up^T              -> silu'(a), h = silu(a)                       (rows F6 of SURVEY.md §8(a))
//   DH  dh = dy[tok] W_down            -> da = g dh silu'(a), hg = g h, dgate = <dh, h>   (rows B1-B3; the gate scales the
//                                         fp32 accumulator in the epilogue instead of the bf16 rows)
//   WG  dW_up = da^T x[tok],  dW_down = dy[tok]^T hg                                   (rows B2, B4: weight gradients)
// One skeleton for all three: a CTA (cta_group::1) owns TWO 128 x 128 fp32 accumulators (or one 128 x 256) in tensor
// memory; per 64-wide K block the GATHERED operand is 32 KB (256 rows x 128 B for F1 / DH, 64 K rows x 512 B for WG) copied
// by 16 warps with 16-byte cp.async into the 128B-swizzle image the tensor core reads, and the other operand is 16 KB
// loaded by TMA; 4 stages of 48 KB.  A gather thread never waits for its data: it waits for a free stage, issues its 4
// copies and lets `cp.async.mbarrier.arrive.noinc` signal the stage's full barrier when they land, so up to 4 stages
// (128 KB per SM) are in flight -- the measured rate of that copy path is ~31 B/clk/SM with 16 warps, above
// what the same rows cost as an HBM round trip through a permuted copy.
//   warp 0: TMA producer of the dense operand     warp 1: MMA issuer (one elected lane, tcgen05.mma M = 128, N = 128 / 256)
//   warp 2: TMEM allocator                        warps 4-7: epilogue (TMEM -> registers -> swizzled tile -> TMA bulk store)
//   warps 8-23: gather
#include <cuda.h>
#include <stdlib.h>

#include "common.cuh"
#include "umma_ptx.cuh"

namespace fomoe {
namespace {

constexpr int GT = 128;                             // rows (columns) of one accumulator tile = d_expert
constexpr int GK = 64;                              // K block
constexpr int kGStages = 4;
constexpr int kGGatherBytes = 2 * GT * GK * 2;      // 32 KB gathered per stage
constexpr int kGTmaBytes = GT * GK * 2;             // 16 KB by TMA
constexpr int kGStageBytes = kGGatherBytes + kGTmaBytes;
constexpr int kGGatherWarps = 16, kGEpiWarps = 4;
constexpr int kGGatherThreads = 32 * kGGatherWarps;
constexpr int kGThreads = 32 * (4 + kGEpiWarps) + kGGatherThreads;   // 768
constexpr int kGStgTile = 2048;                     // 32 rows x 32 bf16, SWIZZLE_64B image of a bulk tensor store
constexpr int kGStgTiles = 4;                       // per epilogue warp: two sets of up to two output tiles
constexpr int kGAccStages = 2, kGTmemCols = 512;    // 2 x (two 128-column accumulators)
constexpr int kGSmem = kGStages * kGStageBytes + kGEpiWarps * kGStgTiles * kGStgTile + 1024 + 256;

enum GMode { G_F1 = 0, G_DH = 1, G_WG = 2 };

struct GMaps {
  // F1: m[0] = W_up (K-major rows), m[1] = silu'(a) out, m[2] = h out
  // DH: m[0] = W_down (MN-major), m[1] = da out, m[2] = hg out
  // WG: m[0] = da, m[1] = hg (both MN-major, K = rows), m[2] = dW_up out, m[3] = dW_down out
  CUtensorMap m[4];
};

struct GParams {
  const int32_t* n_mtiles;     // [2] = row-tile pairs in use
  const int32_t* tile_slot;    // slot of row tile
  const int32_t* pair_info;    // 2 * first row tile + (second tile in the same slot)
  const int32_t* pad_offsets;  // WG: first padded row of slot s
  const int32_t* pad_end64;    // WG: end of slot s's K range
  const int32_t* prow_token;   // token of padded row r, -1 = padding row (gathered as zeros)
  const float* prow_gate;      // DH: gate of padded row r
  const bf16* g0;              // gathered source [T, d]: F1 x, DH dy, WG x (dW_up)
  const bf16* g1;              // WG: dy (dW_down)
  const bf16* in0;             // DH: silu'(a) [R, F]
  const bf16* in_h;            // DH: h [R, F]
  float* dgate_part;           // DH: [R, n_dgate_parts]: part 0 = <dh, h> (not scaled by the gate), the rest 0
  int n_dgate_parts;
  int d, n_res;
  // WG: the tiles of the last, partially filled round of the grid (tile ids >= wg_full; all of them when the tiles do not
  // fill the SMs once) have their K range cut into `ks` parts, each part an item of its own writing an fp32 partial
  // [128, 256] to `part`; fine_wg_reduce_kernel adds them in a fixed order
  int ks, wg_full;
  float* part;
};

__device__ __forceinline__ void g_cp_async16(uint32_t dst, const void* src, bool valid) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(valid ? 16 : 0) : "memory");
}
// the barrier gets one arrival once all cp.async issued so far by this thread have landed (counted in its init value)
__device__ __forceinline__ void g_cp_async_arrive(uint32_t bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void g_tma_load(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
               ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(bar), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void g_mma(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}"
               ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void g_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void g_mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void g_tmem_ld16(uint32_t taddr, float (&v)[16]) {
  uint32_t* r = reinterpret_cast<uint32_t*>(v);
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
                 "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr));
}
__device__ __forceinline__ void g_sts128(uint32_t addr, const uint4& v) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ uint4 g_lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ uint32_t g_pack(float lo, float hi) {
  __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&h);
}
__device__ __forceinline__ float2 g_unpack(uint32_t w) { return __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&w)); }
// lane = row: 16 fp32 as bf16 into 16-byte pieces q0, q0 + 1 of this lane's row of a 32 x 64 B SWIZZLE_64B tile
__device__ __forceinline__ void g_put16(uint32_t stg, int lane, int q0, const float (&v)[16]) {
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    uint4 w;
    w.x = g_pack(v[8 * j + 0], v[8 * j + 1]);
    w.y = g_pack(v[8 * j + 2], v[8 * j + 3]);
    w.z = g_pack(v[8 * j + 4], v[8 * j + 5]);
    w.w = g_pack(v[8 * j + 6], v[8 * j + 7]);
    g_sts128(stg + lane * 64 + (((q0 + j) ^ ((lane >> 1) & 3)) << 4), w);
  }
}
// instruction descriptor: D fp32, A / B bf16, M = 128, N = n, majorness per operand (0 = K-major, 1 = MN-major)
__device__ __forceinline__ constexpr uint32_t g_idesc(int a_mn, int b_mn, int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_mn << 15) | ((uint32_t)b_mn << 16) | ((uint32_t)(n >> 3) << 17) |
         ((uint32_t)(GT >> 4) << 24);
}

// ---------------------------------------------------------------------------------------------------------
// work items.  F1 / DH: the row-tile pairs of the route workspace; the pairs beyond the last full round of the grid are
// handed out as single 128-row tiles so that the tail round takes half a pair's time.  WG: (slot, job, 256-column block).
// ---------------------------------------------------------------------------------------------------------
struct GItem {
  int row0;      // F1 / DH: first padded row.  WG: first row of the slot's K range
  int ntiles;    // F1 / DH: live 128-row tiles (0 = nothing to do).  WG: 2
  int slot;
  int num_kb;
  int job, n0;   // WG: 0 = dW_up (gathered operand = B, N = 256), 1 = dW_down (gathered = A, two 128-row halves); first d column
  long pidx;     // WG split-K: index of this item's partial tile in GParams::part, -1 = a whole tile (stored as bf16)
};

// WG tile numbering (shared with fine_wg_reduce_kernel).  d <= 1024: column block outermost -- neighbouring tiles gather the
// same 256 columns of x / dy for different slots (P2: 62 -> 55 us, P1: 28 -> 27 us).  Wider rows: slot outermost, so that the
// tiles in flight cover whole rows; with the column block outermost every CTA would read the same 512-byte stripe of 4 KB
// rows at once and the kernel slows down although its DRAM traffic drops (P3: 169 -> 196 us, measured).
__device__ __forceinline__ void wg_tile(long id, int n_res, int d, int& slot, int& job, int& n0) {
  const int ntn = d / 256;
  if (ntn <= 4) {
    n0 = (int)(id / (2 * n_res)) * 256;
    const int rem = (int)(id % (2 * n_res));
    slot = rem >> 1;
    job = rem & 1;
  } else {
    slot = (int)(id / (2 * ntn));
    const int rem = (int)(id % (2 * ntn));
    job = rem / ntn;
    n0 = (rem % ntn) * 256;
  }
}

template <int MODE>
struct GSched {
  const GParams& p;
  long total, full;
  __device__ GSched(const GParams& p_, int grid) : p(p_) {
    if (MODE == G_WG) {
      const long tiles = (long)p.n_res * 2 * (p.d / 256);
      full = p.wg_full;
      total = full + (tiles - full) * p.ks;
    } else {
      const long n_pairs = p.n_mtiles[2];
      full = n_pairs / grid * grid;
      total = full + 2 * (n_pairs - full);
    }
  }
  __device__ GItem decode(long id) const {
    GItem it;
    it.job = 0; it.n0 = 0;
    if (MODE == G_WG) {
      it.pidx = -1;
      int kpart = 0;
      if (id >= full) {
        it.pidx = id - full;
        kpart = (int)(it.pidx % p.ks);
        id = full + it.pidx / p.ks;
      }
      wg_tile(id, p.n_res, p.d, it.slot, it.job, it.n0);
      it.row0 = p.pad_offsets[it.slot];
      it.num_kb = (p.pad_end64[it.slot] - it.row0 + GK - 1) / GK;
      if (it.pidx >= 0 && p.ks > 1) {   // this part's K blocks
        const int per = (it.num_kb + p.ks - 1) / p.ks, kb0 = min(kpart * per, it.num_kb), kb1 = min(kb0 + per, it.num_kb);
        it.row0 += kb0 * GK;
        it.num_kb = kb1 - kb0;
      }
      it.ntiles = 2;
    } else {
      int first;
      if (id < full) {
        const int info = p.pair_info[id];
        first = info >> 1;
        it.ntiles = 1 + (info & 1);
        it.slot = p.tile_slot[first];
      } else {
        const long j = id - full;
        const int info = p.pair_info[full + (j >> 1)];
        first = (info >> 1) + (int)(j & 1);
        it.ntiles = ((j & 1) && !(info & 1)) ? 0 : 1;
        it.slot = p.tile_slot[info >> 1];
      }
      it.row0 = first * GT;
      it.num_kb = p.d / GK;
    }
    return it;
  }
};

// ---------------------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(kGThreads, 1)
fine_gather_kernel(const __grid_constant__ GMaps maps, const __grid_constant__ GParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint8_t* stg_base = smem + kGStages * kGStageBytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(stg_base + kGEpiWarps * kGStgTiles * kGStgTile);
  uint64_t* full_bar = bars;                                  // [kGStages]   gather threads + the TMA producer's expect_tx
  uint64_t* empty_bar = bars + kGStages;                      // [kGStages]   released by the MMA issuer's commit
  uint64_t* tfull_bar = bars + 2 * kGStages;                  // [kGAccStages]
  uint64_t* tempty_bar = bars + 2 * kGStages + kGAccStages;   // [kGAccStages] one arrival per epilogue warp
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * kGStages + 2 * kGAccStages);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  pdl_launch_dependents();
  if (warp == 0 && lane == 0) {
#pragma unroll
    for (int i = 0; i < 4; ++i) prefetch_tmap(&maps.m[i]);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < kGStages; ++i) { mbar_init(smem_u32(&full_bar[i]), kGGatherThreads + 1); mbar_init(smem_u32(&empty_bar[i]), 1); }
    for (int i = 0; i < kGAccStages; ++i) { mbar_init(smem_u32(&tfull_bar[i]), 1); mbar_init(smem_u32(&tempty_bar[i]), kGEpiWarps); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(kGTmemCols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  pdl_wait();   // everything below reads what earlier kernels wrote

  const GSched<MODE> sched(p, (int)gridDim.x);
  const uint32_t smem0 = smem_u32(smem);

  if (warp == 0) {
    // ===================== TMA producer: the dense 16 KB operand of every K block =====================
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (long id = blockIdx.x; id < sched.total; id += gridDim.x) {
        const GItem it = sched.decode(id);
        if (it.ntiles == 0) continue;
        for (int kb = 0; kb < it.num_kb; ++kb) {
          mbar_wait(smem_u32(&empty_bar[stage]), phase ^ 1);
          const uint32_t sa = smem0 + stage * kGStageBytes + kGGatherBytes, fb = smem_u32(&full_bar[stage]);
          mbar_expect_tx(fb, kGTmaBytes);
          if (MODE == G_F1) {          // W_up rows [slot F, slot F + 128), K-major: box {64, 128}
            g_tma_load(sa, &maps.m[0], fb, kb * GK, it.slot * GT);
          } else if (MODE == G_DH) {   // W_down [slot d + k, f], MN-major: two {64 columns, 64 rows} boxes
            g_tma_load(sa, &maps.m[0], fb, 0, it.slot * p.d + kb * GK);
            g_tma_load(sa + 8192, &maps.m[0], fb, 64, it.slot * p.d + kb * GK);
          } else {                     // da / hg rows of the K block, MN-major
            g_tma_load(sa, &maps.m[it.job], fb, 0, it.row0 + kb * GK);
            g_tma_load(sa + 8192, &maps.m[it.job], fb, 64, it.row0 + kb * GK);
          }
          if (++stage == kGStages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    int stage = 0, as = 0;
    uint32_t phase = 0, aphase = 0;
    for (long id = blockIdx.x; id < sched.total; id += gridDim.x) {
      const GItem it = sched.decode(id);
      if (it.ntiles == 0 || it.num_kb == 0) continue;   // (empty WG group: the epilogue writes zeros without tensor memory)
      mbar_wait(smem_u32(&tempty_bar[as]), aphase ^ 1);
      const uint32_t tmem_d = tmem_base + as * 256;
      for (int kb = 0; kb < it.num_kb; ++kb) {
        mbar_wait(smem_u32(&full_bar[stage]), phase);
        // the gathered rows were written through the generic proxy (cp.async); the tensor core reads through the async proxy
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        tc_fence_after();
        if (elect_one_sync()) {
          const uint32_t ga = smem0 + stage * kGStageBytes, ta = ga + kGGatherBytes;
          const uint32_t acc0 = kb != 0 ? 1u : 0u;
          if (MODE == G_F1 || MODE == G_DH) {
            // A = gathered rows, K-major (16 K elements = 32 B inside the swizzle row); B: F1 K-major, DH MN-major (16 K rows = 2048 B)
            const uint64_t bdesc = MODE == G_F1 ? make_desc(ta, 16, 1024) : make_desc(ta, 8192, 1024);
            constexpr uint32_t kBStep = MODE == G_F1 ? 2 : 128;
            constexpr uint32_t idesc = g_idesc(0, MODE == G_F1 ? 0 : 1, 128);
            for (int half = 0; half < it.ntiles; ++half) {
              const uint64_t adesc = make_desc(ga + half * 16384, 16, 1024);
#pragma unroll
              for (int k4 = 0; k4 < 4; ++k4) g_mma(tmem_d + half * 128, adesc + 2 * k4, bdesc + kBStep * k4, idesc, k4 ? 1u : acc0);
            }
          } else if (it.job == 0) {   // dW_up [128 f, 256 d columns] = da^T x: A = da (TMA), B = gathered x rows, both MN-major
            const uint64_t adesc = make_desc(ta, 8192, 1024), bdesc = make_desc(ga, 8192, 1024);
            constexpr uint32_t idesc = g_idesc(1, 1, 256);
#pragma unroll
            for (int k4 = 0; k4 < 4; ++k4) g_mma(tmem_d, adesc + 128 * k4, bdesc + 128 * k4, idesc, k4 ? 1u : acc0);
          } else {                    // dW_down [2 x 128 d rows, 128 f] = dy^T hg: A = gathered dy rows, B = hg (TMA)
            const uint64_t bdesc = make_desc(ta, 8192, 1024);
            constexpr uint32_t idesc = g_idesc(1, 1, 128);
#pragma unroll
            for (int half = 0; half < 2; ++half) {
              const uint64_t adesc = make_desc(ga + half * 16384, 8192, 1024);
#pragma unroll
              for (int k4 = 0; k4 < 4; ++k4) g_mma(tmem_d + half * 128, adesc + 128 * k4, bdesc + 128 * k4, idesc, k4 ? 1u : acc0);
            }
          }
          g_commit(smem_u32(&empty_bar[stage]));
          if (kb == it.num_kb - 1) g_commit(smem_u32(&tfull_bar[as]));
        }
        __syncwarp();
        if (++stage == kGStages) { stage = 0; phase ^= 1; }
      }
      if (++as == kGAccStages) { as = 0; aphase ^= 1; }
    }
  } else if (warp >= 4 + kGEpiWarps) {
    // ===================== gather warps =====================
    const int g = threadIdx.x - 32 * (4 + kGEpiWarps);
    int stage = 0;
    uint32_t phase = 0;
    if (MODE == G_F1 || MODE == G_DH) {
      // 256 rows x 8 pieces of 16 B per K block: this thread copies piece c of rows r0, r0 + 64, r0 + 128, r0 + 192
      const int c = g & 7, r0 = g >> 3;
      const uint32_t dst0 = (uint32_t)(r0 * 128 + ((c ^ (r0 & 7)) << 4));
      for (long id = blockIdx.x; id < sched.total; id += gridDim.x) {
        const GItem it = sched.decode(id);
        if (it.ntiles == 0) continue;
        const bf16* src[4];
        bool ok[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int tok = (i >> 1) < it.ntiles ? p.prow_token[it.row0 + r0 + 64 * i] : -1;
          ok[i] = tok >= 0;
          src[i] = p.g0 + (size_t)(ok[i] ? tok : 0) * p.d + c * 8;
        }
        const int n_i = 2 * it.ntiles;
        for (int kb = 0; kb < it.num_kb; ++kb) {
          mbar_wait(smem_u32(&empty_bar[stage]), phase ^ 1);
          const uint32_t dst = smem0 + stage * kGStageBytes + dst0;
#pragma unroll
          for (int i = 0; i < 4; ++i)
            if (i < n_i) g_cp_async16(dst + i * 8192, src[i] + kb * GK, ok[i]);
          g_cp_async_arrive(smem_u32(&full_bar[stage]));
          if (++stage == kGStages) { stage = 0; phase ^= 1; }
        }
      }
    } else {
      // 64 K rows x 32 pieces (512 B = 256 columns) per K block: this thread copies piece pc of rows kr0, kr0 + 16, + 32, + 48
      // into the MN-major image: 64-column chunk (pc / 8) at 8192 B, row at 128 B, piece XOR-swizzled by the row
      const int pc = g & 31, kr0 = g >> 5;
      const uint32_t dst0 = (uint32_t)((pc >> 3) * 8192 + kr0 * 128 + (((pc & 7) ^ (kr0 & 7)) << 4));
      for (long id = blockIdx.x; id < sched.total; id += gridDim.x) {
        const GItem it = sched.decode(id);
        if (it.num_kb == 0) continue;
        const bf16* src = (it.job == 0 ? p.g0 : p.g1) + it.n0 + pc * 8;
        int tok[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) tok[i] = p.prow_token[it.row0 + kr0 + 16 * i];
        for (int kb = 0; kb < it.num_kb; ++kb) {
          mbar_wait(smem_u32(&empty_bar[stage]), phase ^ 1);
          const uint32_t dst = smem0 + stage * kGStageBytes + dst0;
#pragma unroll
          for (int i = 0; i < 4; ++i) g_cp_async16(dst + i * 2048, src + (size_t)(tok[i] >= 0 ? tok[i] : 0) * p.d, tok[i] >= 0);
          g_cp_async_arrive(smem_u32(&full_bar[stage]));
          if (kb + 1 < it.num_kb) {
#pragma unroll
            for (int i = 0; i < 4; ++i) tok[i] = p.prow_token[it.row0 + (kb + 1) * GK + kr0 + 16 * i];
          }
          if (++stage == kGStages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp >= 4) {
    // ===================== epilogue: warp q drains TMEM lanes [32 q, 32 q + 32) of both accumulators =====================
    const int q = warp & 3;
    const uint32_t stg_w = smem_u32(stg_base) + (uint32_t)((warp - 4) * kGStgTiles * kGStgTile);
    int as = 0, nst = 0;
    uint32_t aphase = 0;
    for (long id = blockIdx.x; id < sched.total; id += gridDim.x) {
      const GItem it = sched.decode(id);
      if (it.ntiles == 0) continue;
      const bool have_acc = it.num_kb > 0;
      if (have_acc) { mbar_wait(smem_u32(&tfull_bar[as]), aphase); tc_fence_after(); }
      const uint32_t tacc = tmem_base + ((uint32_t)(q * 32) << 16) + as * 256;
      if (MODE == G_F1) {
        for (int half = 0; half < it.ntiles; ++half) {
          const int rw = it.row0 + half * GT + q * 32;
#pragma unroll 1
          for (int cc = 0; cc < 4; ++cc) {
            const uint32_t s0 = stg_w + (nst & 1) * 2 * kGStgTile, s1 = s0 + kGStgTile;
            if (lane == 0) bulk_wait_read<1>();   // the stores that last read this pair of tiles (two chunks ago) have their data
            __syncwarp();
#pragma unroll
            for (int sub = 0; sub < 2; ++sub) {
              float a[16], h[16];
              g_tmem_ld16(tacc + half * 128 + cc * 32 + sub * 16, a);
              tmem_ld_wait();
#pragma unroll
              for (int i = 0; i < 16; ++i) {
                const float sg = __fdividef(1.0f, 1.0f + __expf(-a[i]));
                h[i] = a[i] * sg;                          // silu(a)
                a[i] = fmaf(h[i], 1.0f - sg, sg);           // silu'(a) = s (1 + a (1 - s))
              }
              g_put16(s0, lane, 2 * sub, a);
              g_put16(s1, lane, 2 * sub, h);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) {
              tma_store_2d(&maps.m[1], s0, cc * 32, rw);
              tma_store_2d(&maps.m[2], s1, cc * 32, rw);
              bulk_commit();
            }
            ++nst;
          }
        }
      } else if (MODE == G_DH) {
        // The saved factors silu'(a) and h of a 32 x 32 chunk are copied (cp.async, each lane its own row's 64 bytes) into
        // the two staging tiles one chunk ahead, overwritten in place with da and hg, and stored from there.
        const int n8 = 4 * it.ntiles;                          // chunks of this item: (half, 32-column block)
        const uint32_t loff = (uint32_t)(lane * 64), lsw = (uint32_t)((lane >> 1) & 3);
        auto issue = [&](int c8) {
          const uint32_t sa = stg_w + (c8 & 1) * 2 * kGStgTile + loff, sh = sa + kGStgTile;
          const size_t off = (size_t)(it.row0 + (c8 >> 2) * GT + q * 32 + lane) * GT + (c8 & 3) * 32;
#pragma unroll
          for (int qq = 0; qq < 4; ++qq) {
            g_cp_async16(sa + ((qq ^ lsw) << 4), p.in0 + off + qq * 8, true);
            g_cp_async16(sh + ((qq ^ lsw) << 4), p.in_h + off + qq * 8, true);
          }
          asm volatile("cp.async.commit_group;" ::: "memory");
        };
        if (lane == 0) bulk_wait_read<0>();   // the previous item's last stores have read the tiles
        __syncwarp();
        issue(0);
        float g = 0.f, dg = 0.f;
        int row = 0;
#pragma unroll 1
        for (int c8 = 0; c8 < n8; ++c8) {
          const int half = c8 >> 2, cc = c8 & 3;
          if (cc == 0) {
            row = it.row0 + half * GT + q * 32 + lane;
            g = p.prow_token[row] >= 0 ? p.prow_gate[row] : 0.f;
            dg = 0.f;                                          // <dy W_down, h> of this lane's row, fixed order
          }
          if (c8 + 1 < n8) {
            if (c8 >= 1) {                                     // the other pair of tiles: chunk c8 - 1's stores must have read it
              if (lane == 0) bulk_wait_read<0>();
              __syncwarp();
            }
            issue(c8 + 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
          } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
          }
          const uint32_t sa = stg_w + (c8 & 1) * 2 * kGStgTile + loff, sh = sa + kGStgTile;
#pragma unroll
          for (int sub = 0; sub < 2; ++sub) {
            float v[16];
            g_tmem_ld16(tacc + half * 128 + cc * 32 + sub * 16, v);
            uint4 wa[2], wh[2];
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              wa[j] = g_lds128(sa + (((2 * sub + j) ^ lsw) << 4));
              wh[j] = g_lds128(sh + (((2 * sub + j) ^ lsw) << 4));
            }
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              uint32_t* ua = reinterpret_cast<uint32_t*>(&wa[j]);
              uint32_t* uh = reinterpret_cast<uint32_t*>(&wh[j]);
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                const float2 a2 = g_unpack(ua[i]), h2 = g_unpack(uh[i]);
                const float d0 = v[8 * j + 2 * i], d1 = v[8 * j + 2 * i + 1];
                dg = fmaf(d0, h2.x, dg);
                dg = fmaf(d1, h2.y, dg);
                ua[i] = g_pack((g * d0) * a2.x, (g * d1) * a2.y);   // da = dh silu'(a), dh = g (dy W_down)
                uh[i] = g_pack(g * h2.x, g * h2.y);                 // the weight gradient's operand: dW_down = dy^T (g h)
              }
              g_sts128(sa + (((2 * sub + j) ^ lsw) << 4), wa[j]);
              g_sts128(sh + (((2 * sub + j) ^ lsw) << 4), wh[j]);
            }
          }
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          __syncwarp();
          if (lane == 0) {
            const int rw = it.row0 + half * GT + q * 32;
            tma_store_2d(&maps.m[1], sa - loff, cc * 32, rw);
            tma_store_2d(&maps.m[2], sh - loff, cc * 32, rw);
            bulk_commit();
          }
          if (cc == 3) {
            float* dp = p.dgate_part + (size_t)row * p.n_dgate_parts;
            dp[0] = dg;
            for (int i = 1; i < p.n_dgate_parts; ++i) dp[i] = 0.f;
          }
        }
      } else {
        // job 0: rows = f, 8 chunks of 32 d columns; job 1: two halves of 128 d rows, 4 chunks of 32 f columns each
        const int n_chunks = 8;
        if (it.pidx >= 0 && p.ks > 1) {   // fp32 partial of this K part: row-per-lane 64-byte segments (tail tiles only)
          float* dst = p.part + ((size_t)it.pidx * GT + q * 32 + lane) * 256;
#pragma unroll 1
          for (int c16 = 0; c16 < 16; ++c16) {
            float v[16];
            if (have_acc) {
              g_tmem_ld16(tacc + c16 * 16, v);
              tmem_ld_wait();
            } else {
#pragma unroll
              for (int i = 0; i < 16; ++i) v[i] = 0.f;
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) reinterpret_cast<float4*>(dst + c16 * 16)[i] = make_float4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
          }
        } else
#pragma unroll 1
        for (int ch = 0; ch < n_chunks; ++ch) {
          const uint32_t s0 = stg_w + (nst & 1) * 2 * kGStgTile;
          if (lane == 0) bulk_wait_read<1>();
          __syncwarp();
#pragma unroll
          for (int sub = 0; sub < 2; ++sub) {
            float v[16];
            if (have_acc) {
              g_tmem_ld16(tacc + ch * 32 + sub * 16, v);   // (job 1: columns [128 half, +128) are the second accumulator)
              tmem_ld_wait();
            } else {
#pragma unroll
              for (int i = 0; i < 16; ++i) v[i] = 0.f;
            }
            g_put16(s0, lane, 2 * sub, v);
          }
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          __syncwarp();
          if (lane == 0) {
            if (it.job == 0) tma_store_2d(&maps.m[2], s0, it.n0 + ch * 32, it.slot * GT + q * 32);
            else tma_store_2d(&maps.m[3], s0, (ch & 3) * 32, it.slot * p.d + it.n0 + (ch >> 2) * GT + q * 32);
            bulk_commit();
          }
          ++nst;
        }
      }
      if (have_acc) {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) g_mbar_arrive(smem_u32(&tempty_bar[as]));
        if (++as == kGAccStages) { as = 0; aphase ^= 1; }
      }
    }
    if (lane == 0) bulk_wait_all();   // shared memory stays valid until the stores have read it
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kGTmemCols) : "memory");
}

// adds the ks partials of every split WG tile in a fixed order and writes dW_up / dW_down as bf16.  grid = (split tiles, 8 row slabs)
__global__ void __launch_bounds__(256)
fine_wg_reduce_kernel(const float* __restrict__ part, int ks, int first_tile, int n_res, int d, bf16* __restrict__ dw_up, bf16* __restrict__ dw_down) {
  pdl_launch_dependents();
  pdl_wait();
  int slot, job, n0;
  wg_tile(first_tile + blockIdx.x, n_res, d, slot, job, n0);
  for (int e = blockIdx.y * 16 * 256 + threadIdx.x * 4; e < (blockIdx.y + 1) * 16 * 256; e += 256 * 4) {
    const int r = e >> 8, c = e & 255;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int j = 0; j < ks; ++j) {
      const float4 v = *reinterpret_cast<const float4*>(part + (((size_t)blockIdx.x * ks + j) * GT + r) * 256 + c);
      acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    uint2 o;
    o.x = g_pack(acc.x, acc.y);
    o.y = g_pack(acc.z, acc.w);
    bf16* dst = job == 0 ? dw_up + ((size_t)slot * GT + r) * d + n0 + c
                         : dw_down + ((size_t)slot * d + n0 + (c >> 7) * GT + r) * GT + (c & 127);
    *reinterpret_cast<uint2*>(dst) = o;
  }
}

template <int MODE>
int g_launch(const GMaps& maps, const GParams& p, cudaStream_t st, const char* name) {
  static PerDeviceOnce attr;
  if (attr.need()) {
    FOMOE_CUDA_OK(cudaFuncSetAttribute(fine_gather_kernel<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGSmem));
    attr.set();
  }
  FOMOE_CUDA_OK(launch_pdl(fine_gather_kernel<MODE>, num_sms(), kGThreads, kGSmem, st, maps, p));
  FOMOE_LAUNCH_OK(name);
  return FOMOE_OK;
}

GParams base_params(const fomoe_config& c, int n_res, const RouteWs& rws) {
  GParams p{};
  p.n_mtiles = rws.n_mtiles; p.tile_slot = rws.tile_slot; p.pair_info = rws.pair_info; p.pad_offsets = rws.pad_offsets;
  p.pad_end64 = rws.pad_end64; p.prow_token = rws.prow_token; p.prow_gate = rws.prow_gate;
  p.d = c.d_model; p.n_res = n_res; p.ks = 1; p.wg_full = 0;
  return p;
}

}  // namespace

// FOMOE_FINE in the environment: bit 0 = F1, bit 1 = DH, bit 2 = WG (needs bit 1: hg comes out of the gathered DH); default all.
int fine_mask(const fomoe_config& c) {
  static const int env = [] { const char* e = getenv("FOMOE_FINE"); return e ? atoi(e) : 7; }();
  if (c.dtype != FOMOE_BF16 || c.expert_fn != FOMOE_EXPERT_SILU || c.d_ff != GT || c.d_model % 256 != 0 || c.T <= 0) return 0;
  int m = env & 7;
  if (!(m & 2)) m &= ~4;
  return m;
}

// a = x[token(r)] W_up^T per padded row r; aws.a <- silu'(a), aws.h <- silu(a)
int fine_fwd1(const fomoe_config& c, int n_res, const void* x, const RouteWs& rws, const ActWs& aws, const void* w_up, cudaStream_t st) {
  const uint64_t R = (uint64_t)rws.R_cap;
  GMaps m{};
  MAP_OK(make_map(&m.m[0], w_up, c.d_model, (uint64_t)n_res * GT, c.d_model, 128));
  MAP_OK(make_map_box(&m.m[1], aws.a, GT, R, GT, 32, 32, CU_TENSOR_MAP_SWIZZLE_64B));
  MAP_OK(make_map_box(&m.m[2], aws.h, GT, R, GT, 32, 32, CU_TENSOR_MAP_SWIZZLE_64B));
  m.m[3] = m.m[0];
  GParams p = base_params(c, n_res, rws);
  p.g0 = (const bf16*)x;
  return g_launch<G_F1>(m, p, st, "fine_gather_kernel<F1>");
}

// dh = dy[token(r)] W_down; sws.da <- g dh silu'(a), hg <- g h, sws.dgate_part[r, 0] <- <dh, h>
int fine_dh(const fomoe_config& c, int n_res, const void* dy, const RouteWs& rws, const ActWs& aws, const ScratchWs& sws, void* hg,
            const void* w_down, cudaStream_t st) {
  const uint64_t R = (uint64_t)rws.R_cap;
  GMaps m{};
  MAP_OK(make_map(&m.m[0], w_down, GT, (uint64_t)n_res * c.d_model, GT, 64));
  MAP_OK(make_map_box(&m.m[1], sws.da, GT, R, GT, 32, 32, CU_TENSOR_MAP_SWIZZLE_64B));
  MAP_OK(make_map_box(&m.m[2], hg, GT, R, GT, 32, 32, CU_TENSOR_MAP_SWIZZLE_64B));
  m.m[3] = m.m[0];
  GParams p = base_params(c, n_res, rws);
  p.g0 = (const bf16*)dy;
  p.in0 = (const bf16*)aws.a; p.in_h = (const bf16*)aws.h;
  p.dgate_part = sws.dgate_part; p.n_dgate_parts = sws.n_dgate_parts;
  return g_launch<G_DH>(m, p, st, "fine_gather_kernel<DH>");
}

// dW_up[s] = da^T x[token(r)], dW_down[s] = dy[token(r)]^T hg over the padded rows r of slot s
int fine_wgrad(const fomoe_config& c, int n_res, const void* x, const void* dy, const RouteWs& rws, const ScratchWs& sws, const void* hg,
               void* dw_up, void* dw_down, cudaStream_t st) {
  const uint64_t R = (uint64_t)rws.R_cap;
  GMaps m{};
  MAP_OK(make_map(&m.m[0], sws.da, GT, R, GT, 64));
  MAP_OK(make_map(&m.m[1], hg, GT, R, GT, 64));
  MAP_OK(make_map_box(&m.m[2], dw_up, c.d_model, (uint64_t)n_res * GT, c.d_model, 32, 32, CU_TENSOR_MAP_SWIZZLE_64B));
  MAP_OK(make_map_box(&m.m[3], dw_down, GT, (uint64_t)n_res * c.d_model, GT, 32, 32, CU_TENSOR_MAP_SWIZZLE_64B));
  GParams p = base_params(c, n_res, rws);
  p.g0 = (const bf16*)x; p.g1 = (const bf16*)dy;
  // tiles that do not fill the SMs once (P1: 32): cut K so that the items do; the partials live where the scaled copy of dy
  // would (unused on this path).  The kernel can split the last round of a longer schedule too (wg_full > 0; P3: 68 of 512
  // tiles, kernel 176 -> 162 us) but the step does not get faster: the router's backward chain on the side stream runs on
  // the SMs that round leaves idle, so only the single-round case is split.
  const int tiles = n_res * 2 * (c.d_model / 256), grid = num_sms();
  const int full = tiles / grid * grid, tail = tiles - full;
  static const bool split_tail_round = getenv("FOMOE_FINE_TAILSPLIT") != nullptr;   // (A/B measurements of the multi-round case)
  int ks = (tail > 0 && (full == 0 || split_tail_round)) ? grid / tail : 1;
  if (ks > 8) ks = 8;
  while (ks > 1 && (size_t)tail * ks * GT * 256 * sizeof(float) > sizeof(bf16) * (size_t)R * c.d_model) --ks;
  p.wg_full = ks > 1 ? full : tiles;
  if (ks > 1) { p.ks = ks; p.part = (float*)sws.dop; }
  int rc = g_launch<G_WG>(m, p, st, "fine_gather_kernel<WG>");
  if (rc != FOMOE_OK || ks <= 1) return rc;
  FOMOE_CUDA_OK(launch_pdl(fine_wg_reduce_kernel, dim3(tail, 8), 256, 0, st, (const float*)p.part, ks, full, n_res, c.d_model, (bf16*)dw_up, (bf16*)dw_down));
  FOMOE_LAUNCH_OK("fine_wg_reduce_kernel");
  return FOMOE_OK;
}

}  // namespace fomoe
