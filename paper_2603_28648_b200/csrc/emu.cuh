// Ozaki-emulated FP64 GEMM on the INT8 tensor cores (
// DESIGN.md reading s12): slice-and-pack kernel (row a4 of section 8(a)) and the tcgen05 / TMEM GEMM.
//
//   a_ik ~ X_ik 2^(e_i - (8 kappa - 2)),  X = sum_s d_s 2^(8 (kappa - s)),  d_s balanced digits in [-128, 127]
//   C_ij = 2^(eA_i + eB_j - 2 (8 kappa - 2)) sum_c P_c 2^(16 kappa - 8 c),   P_c = sum_{s+t=c} d^A_s d^B_t (INT32)
//
// Sliced operands are stored K-major, [slice][line][Kpad] int8 with lines padded to the tile and Kpad a
// multiple of 32 (zero filled), so a 32-deep K step of a line is two aligned 16-byte chunks that cp.async
// drops into the no-swizzle UMMA layout of tc_i8.cuh.  The kappa anti-diagonal accumulators (triangular
// product set, s + t <= kappa + 1) live side by side in TMEM: kappa * 64 <= 448 columns.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "tc_i8.cuh"

namespace dmrg {

static constexpr int EMU_BM = 128, EMU_BN = 64, EMU_KS = 32, EMU_STAGES = 4, EMU_MAX_KAPPA = 7;

// One CTA per (line, K chunk) (a row of A or a column of B): exponent e = frexp exponent of max |a| over
// the chunk, then X = rint(a 2^(8 kappa - 2 - e)) and its balanced base-256 digits, top digit in slice 0.
// Exponents are stored as expo[chunk * lines_pad + line]  (Appendix A6: exponents are per K chunk).
__global__ void __launch_bounds__(128) k_emu_slice(const double *__restrict__ src, int n_lines, int Ktot, int64_t line_stride,
                                                   int64_t k_stride, int kappa, int8_t *__restrict__ out,
                                                   int64_t lines_pad, int64_t Kpad, int32_t *__restrict__ expo,
                                                   int kchunk) {
  const int line = blockIdx.x, k_begin = blockIdx.y * kchunk;
  if (line >= n_lines) return;
  const int K = min(kchunk, Ktot - k_begin);
  const double *p = src + (int64_t)line * line_stride + (int64_t)k_begin * k_stride;
  out += k_begin;
  expo += (int64_t)blockIdx.y * lines_pad;
  __shared__ double red[4];
  double mx = 0.0;
  for (int k = threadIdx.x; k < K; k += 128) mx = fmax(mx, fabs(p[(int64_t)k * k_stride]));
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mx;
  __syncthreads();
  mx = fmax(fmax(red[0], red[1]), fmax(red[2], red[3]));
  int e = 0;
  if (mx > 0.0) frexp(mx, &e);
  if (threadIdx.x == 0) expo[line] = e;
  const int sh = 8 * kappa - 2 - e;
  for (int k = threadIdx.x; k < K; k += 128) {
    long long r = llrint(scalbn(p[(int64_t)k * k_stride], sh));
    int8_t *o = out + (int64_t)line * Kpad + k;
    for (int s = kappa - 1; s >= 1; --s) {
      long long d = ((r + 128) & 255) - 128;       // balanced digit in [-128, 127]
      o[(int64_t)s * lines_pad * Kpad] = (int8_t)d;
      r = (r - d) >> 8;                            // exact: r - d is a multiple of 256
    }
    o[0] = (int8_t)r;
  }
}

// C[M][N] (row-major, ldc) = A B from the sliced operands.  grid = (ceil(M/128), ceil(N/64)), 128 threads:
// warp 0 issues the tcgen05 MMAs (one elected lane), warps 1-3 are the cp.async producers, and all four warps
// drain TMEM in the epilogue of every K chunk (warp w owns TMEM lanes 32 w .. 32 w + 31 = rows of the tile).
// Producer -> MMA: mbarrier full[stage] (96 arrivals, after cp.async.wait_group + fence.proxy.async);
// MMA -> producer: tcgen05.commit on empty[stage]; MMA -> epilogue: tcgen05.commit on `done`.
// asl: [kappa][Mpad][Kpad], bsl: [kappa][Npad][Kpad]; K is processed in chunks of at most kchunk (a multiple
// of 32) so that the INT32 accumulators cannot overflow; chunks are summed in FP64 registers.
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"((uint32_t)__cvta_generic_to_shared(bar)) : "memory");
}

template <int KAPPA>
__global__ void __launch_bounds__(128) k_emu_gemm(const int8_t *__restrict__ asl, const int8_t *__restrict__ bsl,
                                                  const int32_t *__restrict__ ea, const int32_t *__restrict__ eb,
                                                  double *__restrict__ C, int M, int N, int64_t ldc, int64_t Mpad,
                                                  int64_t Npad, int64_t Kpad, int kchunk) {
  constexpr int A_SLICE = 2 * EMU_BM * 16, B_SLICE = 2 * EMU_BN * 16, STAGE = KAPPA * (A_SLICE + B_SLICE);
  constexpr int N_PROD = 96, COPIES = KAPPA * 2 * (EMU_BM + EMU_BN);   // 16-byte copies per K step
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ __align__(8) uint64_t bar_full[EMU_STAGES], bar_empty[EMU_STAGES], bar_done;
  __shared__ uint32_t tmem_slot;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int m0 = blockIdx.x * EMU_BM, n0 = blockIdx.y * EMU_BN;
  const uint32_t smem_base = (uint32_t)__cvta_generic_to_shared(smem);

  if (warp == 0) tmem_alloc(&tmem_slot, 512);
  if (tid == 0) {
    for (int s = 0; s < EMU_STAGES; ++s) { mbar_init(&bar_full[s], N_PROD); mbar_init(&bar_empty[s], 1); }
    mbar_init(&bar_done, 1);
  }
  asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const uint32_t tmem = tmem_slot;

  double facc[EMU_BN];
#pragma unroll
  for (int j = 0; j < EMU_BN; ++j) facc[j] = 0.0;
  const int row = m0 + tid;
  const int total_steps = (int)(Kpad / EMU_KS), steps_per_chunk = kchunk / EMU_KS;
  uint32_t full_phase = 0, empty_phase = 0, done_phase = 0;   // bit s: parity to wait for next on stage s
  int step0 = 0;                                              // first K step of the current chunk
  int use = 0;                                                // global count of stage uses (same in every role)

  for (int chunk = 0; step0 < total_steps; ++chunk, step0 += steps_per_chunk) {
    const int nsteps = min(steps_per_chunk, total_steps - step0);
    if (warp == 0) {
      // ---------------- MMA issuer
      if (lane == 0) {
        const uint32_t idesc = umma_idesc_s8(EMU_BM, EMU_BN);
        for (int k = 0; k < nsteps; ++k) {
          const int st = (use + k) % EMU_STAGES;
          mbar_wait(&bar_full[st], (full_phase >> st) & 1u); full_phase ^= 1u << st;
          asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
          const uint32_t sa = smem_base + st * STAGE, sb = sa + KAPPA * A_SLICE;
          const uint64_t da = umma_smem_desc(sa, EMU_BM * 16, 128), db = umma_smem_desc(sb, EMU_BN * 16, 128);
#pragma unroll
          for (int s = 0; s < KAPPA; ++s)
#pragma unroll
            for (int t = 0; s + t < KAPPA; ++t)      // triangular set: (s+1) + (t+1) <= kappa + 1
              umma_i8(tmem + (uint32_t)((s + t) * EMU_BN), da + (uint64_t)((s * A_SLICE) >> 4),
                      db + (uint64_t)((t * B_SLICE) >> 4), idesc, !(k == 0 && s == 0));   // the first product of an anti-diagonal overwrites
          umma_commit(&bar_empty[st]);
        }
        umma_commit(&bar_done);
      }
      __syncwarp();
    } else {
      // ---------------- producers: 96 threads, two K steps in flight before signalling
      const int p = tid - 32;
      for (int k = 0; k < nsteps + 2; ++k) {
        if (k < nsteps) {
          const int st = (use + k) % EMU_STAGES;
          if (use + k >= EMU_STAGES) { mbar_wait(&bar_empty[st], (empty_phase >> st) & 1u); empty_phase ^= 1u << st; }
          const uint32_t sa = smem_base + st * STAGE, sb = sa + KAPPA * A_SLICE;
          const int64_t kbyte = (int64_t)(step0 + k) * EMU_KS;
          for (int i = p; i < COPIES; i += N_PROD) {
            if (i < KAPPA * 2 * EMU_BM) {
              const int r = i % EMU_BM, c = (i / EMU_BM) & 1, s = i / (2 * EMU_BM);
              const int8_t *g = asl + ((int64_t)s * Mpad + m0 + r) * Kpad + kbyte + c * 16;
              asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa + s * A_SLICE + (c * EMU_BM + r) * 16), "l"(g));
            } else {
              const int i2 = i - KAPPA * 2 * EMU_BM;
              const int r = i2 % EMU_BN, c = (i2 / EMU_BN) & 1, s = i2 / (2 * EMU_BN);
              const int8_t *g = bsl + ((int64_t)s * Npad + n0 + r) * Kpad + kbyte + c * 16;
              asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sb + s * B_SLICE + (c * EMU_BN + r) * 16), "l"(g));
            }
          }
        }
        cp_async_commit();
        if (k >= 2) {                              // the copies of step k - 2 have landed
          cp_async_wait<2>();
          asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
          mbar_arrive(&bar_full[(use + k - 2) % EMU_STAGES]);
        }
      }
    }
    use += nsteps;
    // ---------------- epilogue of the chunk: TMEM -> registers, FP64, smallest scale first
    mbar_wait(&bar_done, done_phase); done_phase ^= 1u;
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    const int e_row = row < M ? __ldg(ea + (int64_t)chunk * Mpad + row) : 0;
#pragma unroll
    for (int c0 = 0; c0 < EMU_BN; c0 += 8) {
      double v[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) v[e] = 0.0;
#pragma unroll
      for (int c = KAPPA - 1; c >= 0; --c) {
        int32_t pv[8];
        tmem_ld8(tmem + ((uint32_t)(warp * 32) << 16) + (uint32_t)(c * EMU_BN + c0), pv);
        const double w = scalbn(1.0, 16 * KAPPA - 8 * (c + 2));
#pragma unroll
        for (int e = 0; e < 8; ++e) v[e] += (double)pv[e] * w;
      }
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        const int col = n0 + c0 + e;
        const int eb_col = col < N ? __ldg(eb + (int64_t)chunk * Npad + col) : 0;
        facc[c0 + e] += scalbn(v[e], e_row + eb_col - 2 * (8 * KAPPA - 2));
      }
    }
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();               // every warp has drained TMEM before the next chunk overwrites it
  }
  if (row < M) {
#pragma unroll
    for (int j = 0; j < EMU_BN; ++j)
      if (n0 + j < N) C[(int64_t)row * ldc + n0 + j] = facc[j];
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 512);
}

}  // namespace dmrg
