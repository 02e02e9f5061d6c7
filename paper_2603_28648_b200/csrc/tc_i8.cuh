// tcgen05 / TMEM INT8 building blocks (sm_100a): the tensor path of the Ozaki-emulated FP64 mode
// (FP64 emulation over fixed-point INT8 slices; SURVEY.md section 7 "Hard parts").
// This file holds the descriptor encodings, the issue / commit / TMEM-load wrappers and k_peak_i8, a
// full-tile kernel that (a) checks one 128 x 256 x 32 s8 MMA element by element against the integer
// definition and (b) measures the sustained INT8 tensor-pipe rate that bench.py reports as P_INT8.
//
// Shared-memory operand layout used here (K-major, no swizzle, "interleave"): for every 16-byte K chunk c
// a column of rows, address = c * (rows * 16) + row * 16.  In UMMA terms: core matrix = 8 rows x 16 B
// (128 contiguous bytes), SBO = 128 B between 8-row groups, LBO = rows * 16 B between K chunks.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace dmrg {

__device__ __forceinline__ uint64_t umma_smem_desc(uint32_t smem_addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr >> 4) & 0x3fff);            // start address, bits [0,14)
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3fff) << 16;      // leading byte offset, bits [16,30)
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3fff) << 32;      // stride byte offset, bits [32,46)
  d |= (uint64_t)1 << 46;                                // descriptor version 1 (sm_100)
  return d;                                              // base offset 0, layout type 0 = no swizzle
}
// kind::i8 instruction descriptor: D = S32, A = B = signed 8 bit, both K-major, dense
__host__ __device__ constexpr uint32_t umma_idesc_s8(int M, int N) {
  return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, bool acc) {
  asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n"
               " tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n}\n"
               ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"((uint32_t)acc) : "memory");
}
// One lane of a converged warp (the same lane at every call with the full mask).  The MMA warp runs its loops with all
// lanes so that descriptors and loop state are provably warp-uniform and live in uniform registers; only the
// tcgen05.mma / tcgen05.commit instructions are predicated on the leader (an `if (lane == 0)` around the whole loop
// makes ptxas wrap every UTCIMMA in an ELECT / R2UR.BROADCAST / BRA.U.ANY loop of ~17 instructions).
__device__ __forceinline__ bool elect_one() {
  uint32_t p;
  asm volatile("{\n .reg .pred q;\n elect.sync _|q, 0xffffffff;\n selp.u32 %0, 1, 0, q;\n}\n" : "=r"(p));
  return p != 0;
}
__device__ __forceinline__ void umma_commit(uint64_t *bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n"
               ::"r"((uint32_t)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile("{\n .reg .pred p;\n WAIT_%=:\n"
               " mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
               " @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n"
               ::"r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tmem_alloc(uint32_t *slot_in_smem, int cols) {   // one full warp
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n"
               ::"r"((uint32_t)__cvta_generic_to_shared(slot_in_smem)), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t addr, int cols) {            // the allocating warp
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(addr), "r"(cols) : "memory");
}
// 32 lanes x 8 consecutive 32-bit columns: thread t of warp w reads lane 32 w + t
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, int32_t (&v)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
               : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
}

// Full-tile INT8 kernel: one CTA per SM, all 512 TMEM columns (two 128 x 256 S32 accumulators).
// A[m][k] = ((3 m + 5 k) mod 11) - 5, B[n][k] = ((7 n + k) mod 9) - 4, k < 32.
// n_mma MMAs alternate between the accumulators; `out` (if non-null, first CTA) receives accumulator 0.
template <int N>
__global__ void __launch_bounds__(128) k_peak_i8(int n_mma, int32_t *out) {
  constexpr int M = 128;
  __shared__ __align__(128) int8_t sA[2 * M * 16];
  __shared__ __align__(128) int8_t sB[2 * N * 16];
  __shared__ __align__(8) uint64_t bar;
  __shared__ uint32_t tmem_slot;
  const int tid = threadIdx.x, warp = tid >> 5;
  for (int i = tid; i < 2 * M * 16; i += 128) {
    int c = i / (M * 16), m = (i / 16) % M, k = c * 16 + (i % 16);
    sA[i] = (int8_t)(((3 * m + 5 * k) % 11) - 5);
  }
  for (int i = tid; i < 2 * N * 16; i += 128) {
    int c = i / (N * 16), n = (i / 16) % N, k = c * 16 + (i % 16);
    sB[i] = (int8_t)(((7 * n + k) % 9) - 4);
  }
  if (warp == 0) tmem_alloc(&tmem_slot, 512);
  if (tid == 0) mbar_init(&bar, 1);
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");       // st.shared -> tensor-core reads
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const uint32_t tmem = tmem_slot;
  if (tid == 0) {
    const uint64_t ad = umma_smem_desc((uint32_t)__cvta_generic_to_shared(sA), M * 16, 128);
    const uint64_t bd = umma_smem_desc((uint32_t)__cvta_generic_to_shared(sB), N * 16, 128);
    const uint32_t idesc = umma_idesc_s8(M, N);
    for (int j = 0; j < n_mma; ++j) umma_i8(tmem + (uint32_t)((j & 1) * 256), ad, bd, idesc, j >= 2);
    umma_commit(&bar);
  }
  mbar_wait(&bar, 0);
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  if (out != nullptr && blockIdx.x == 0) {
    for (int c0 = 0; c0 < N; c0 += 8) {
      int32_t v[8];
      tmem_ld8(tmem + ((uint32_t)(warp * 32) << 16) + (uint32_t)c0, v);
      for (int e = 0; e < 8; ++e) out[(size_t)tid * N + c0 + e] = v[e];
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 512);
}

}  // namespace dmrg
