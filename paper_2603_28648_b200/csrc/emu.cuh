// Ozaki-emulated FP64 GEMM on the INT8 tensor cores (
// DESIGN.md reading s12): slice-and-pack kernel (row a4 of section 8(a)) and the tcgen05 / TMEM GEMM.
//
//   a_ik ~ X_ik 2^(e_i - (8 kappa - 2)),  X = sum_s d_s 2^(8 (kappa - s)),  d_s balanced digits in [-128, 127]
//   C_ij = 2^(eA_i + eB_j - 2 (8 kappa - 2)) sum_c P_c 2^(16 kappa - 8 c),   P_c = sum_{s+t=c} d^A_s d^B_t (INT32)
//
// This file holds the constants and the plain slicing kernel behind dmrg_emu_slice ([slice][line][K] output,
// the layout the bit-exact digit tests read); the engine itself (pre-tiled slices, bulk-copy pipeline,
// persistent tcgen05 kernel) is in emu_seg.cuh.  The kappa anti-diagonal accumulators (triangular product
// set, s + t <= kappa + 1) live side by side in TMEM: kappa * 64 <= 448 columns.
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

}  // namespace dmrg
