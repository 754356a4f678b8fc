// Resident-delta pack (row S1 of SURVEY.md §8(a)): payload = w_start - w_now per resident expert, fp32, laid out as
// per-expert blocks [gate | up | down] (PAPER.md:253 payload content; 824 Alg. 2 l.19; 163 Fig. 4 one ring per expert).
// Pure streaming: 12 bytes of HBM traffic per parameter (two fp32 reads, one fp32 write), 16-byte vectors, loads
// bypass L1 and evict first, 4 independent vectors per thread in flight.
#include "common.cuh"

namespace fomoe {

struct f8 { float v[8]; };
// 32-byte vector accesses (sm_100: ld/st.global.v8.b32), streaming: no L1 allocation, L2 evict-first.
__device__ __forceinline__ f8 ld_stream(const f8* p) {
  f8 r;
  uint32_t* u = reinterpret_cast<uint32_t*>(r.v);
  asm volatile("ld.global.nc.L1::no_allocate.L2::evict_first.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]), "=r"(u[6]), "=r"(u[7]) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream(f8* p, const f8& r) {
  const uint32_t* u = reinterpret_cast<const uint32_t*>(r.v);
  asm volatile("st.global.L1::no_allocate.L2::evict_first.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(u[0]), "r"(u[1]),
               "r"(u[2]), "r"(u[3]), "r"(u[4]), "r"(u[5]), "r"(u[6]), "r"(u[7]) : "memory");
}
struct f4 { float v[4]; };
__device__ __forceinline__ f4 ld_stream(const f4* p) {
  f4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream(f4* p, const f4& r) {
  asm volatile("st.global.cs.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(r.v[0]), "f"(r.v[1]), "f"(r.v[2]), "f"(r.v[3]) : "memory");
}

struct PackArgs {
  const float* now[3];
  const float* start[3];
  long nvec[3];     // vectors per slot of each tensor
  long out_off[3];  // vector offset of each tensor inside a payload block
  long block_vec;   // vectors per payload block
};

constexpr int kPackThreads = 256, kPackUnroll = 4;

// grid: (x: strided chunks, y: packed slot b, z: tensor).  VT = f8 (32-byte vectors) or f4 (16-byte).
template <typename VT>
__global__ void __launch_bounds__(kPackThreads)
pack_kernel(PackArgs a, const int32_t* __restrict__ pack_slots, float* __restrict__ payload) {
  constexpr int W = sizeof(VT) / 4;
  const int b = blockIdx.y, z = blockIdx.z;
  const int s = pack_slots ? pack_slots[b] : b;
  const long n = a.nvec[z];
  const VT* __restrict__ now = reinterpret_cast<const VT*>(a.now[z]) + (size_t)s * n;
  const VT* __restrict__ start = reinterpret_cast<const VT*>(a.start[z]) + (size_t)s * n;
  VT* __restrict__ out = reinterpret_cast<VT*>(payload) + (size_t)b * a.block_vec + a.out_off[z];
  const long stride = (long)gridDim.x * kPackThreads * kPackUnroll;
  for (long base = (long)blockIdx.x * kPackThreads * kPackUnroll + threadIdx.x; base < n; base += stride) {
    VT w0[kPackUnroll], w1[kPackUnroll];
#pragma unroll
    for (int u = 0; u < kPackUnroll; ++u) {
      long i = base + (long)u * kPackThreads;
      if (i < n) { w1[u] = ld_stream(start + i); w0[u] = ld_stream(now + i); }
    }
#pragma unroll
    for (int u = 0; u < kPackUnroll; ++u) {
      long i = base + (long)u * kPackThreads;
      if (i < n) {
        VT r;
#pragma unroll
        for (int q = 0; q < W; ++q) r.v[q] = w1[u].v[q] - w0[u].v[q];
        st_stream(out + i, r);
      }
    }
  }
}

int launch_pack(const float* const w_now[3], const float* const w_start[3], int n_res, int64_t eg, int64_t eu, int64_t ed,
                const int32_t* pack_slots, int n_pack, float* payload, cudaStream_t st) {
  (void)n_res;
  if (n_pack == 0) return FOMOE_OK;
  const int64_t e[3] = {eg, eu, ed};
  bool wide = (reinterpret_cast<uintptr_t>(payload) & 31u) == 0;
  for (int i = 0; i < 3; ++i)
    wide = wide && e[i] % 8 == 0 && (reinterpret_cast<uintptr_t>(w_now[i]) & 31u) == 0 && (reinterpret_cast<uintptr_t>(w_start[i]) & 31u) == 0;
  const int W = wide ? 8 : 4;
  PackArgs a;
  long off = 0, maxvec = 0;
  for (int i = 0; i < 3; ++i) {
    a.now[i] = w_now[i];
    a.start[i] = w_start[i];
    a.nvec[i] = (long)(e[i] / W);
    a.out_off[i] = off;
    off += a.nvec[i];
    if (a.nvec[i] > maxvec) maxvec = a.nvec[i];
  }
  a.block_vec = off;
  const long per_block = (long)kPackThreads * kPackUnroll;
  long gx = (maxvec + per_block - 1) / per_block;
  // ~16 CTAs per SM in total keeps enough bytes in flight
  long want = ((long)num_sms() * 16 + (long)n_pack * 3 - 1) / ((long)n_pack * 3);
  if (gx > want) gx = want;
  if (gx < 1) gx = 1;
  dim3 grid((unsigned)gx, (unsigned)n_pack, 3);
  if (wide) pack_kernel<f8><<<grid, kPackThreads, 0, st>>>(a, pack_slots, payload);
  else pack_kernel<f4><<<grid, kPackThreads, 0, st>>>(a, pack_slots, payload);
  FOMOE_LAUNCH_OK("pack_kernel");
  return FOMOE_OK;
}

}  // namespace fomoe
