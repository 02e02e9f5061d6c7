// Emulated-FP64 stage 2 of H_eff.psi (DMRG_PREC_FP64_EMU): descriptor-driven slice-and-pack (row a4) for
// the class-stacked left operators (once per bond) and for the intermediate T (every apply), and the
// segmented tcgen05 INT8 kernel that accumulates psi'[b'] = sum_seg G_seg O_L,seg T_seg with one exponent
// set per segment (SURVEY.md section 7 "Hard parts" 2-5, Appendix A6).
//
// Sliced layout of one operand block: [slice][line][K], K = member * dlpad + l with dlpad = roundup(dl, 32)
// (zero filled), so a segment (a member range) is an aligned K range and a 32-deep K step of a line is two
// 16-byte chunks.  Exponents are per line over the whole block (operators) or the whole stage-1 job (T).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "emu.cuh"

namespace dmrg {

__device__ __forceinline__ void emu_digits(double x, int sh, int kappa, int8_t *d) {   // top digit in d[0]
  long long r = llrint(scalbn(x, sh));
  for (int s = kappa - 1; s >= 1; --s) {
    long long q = ((r + 128) & 255) - 128;
    d[s] = (int8_t)q;
    r = (r - q) >> 8;
  }
  d[0] = (int8_t)r;
}

// grid = (descriptors, line tiles), 256 threads.  element(line, member, l) = src + member*mstride + l*lstride
// + line*linestride.  Lines are processed 32 at a time; the thread block is 32 (fast index) x 8.
//   linestride == 1: threads run along lines when reading (coalesced), digits are transposed through shared
//                    memory so that the int8 output is written along K;
//   otherwise (lstride == 1): threads run along l when reading.
__global__ void __launch_bounds__(256) k_emu_slice_desc(const EmuSliceDesc *__restrict__ descs, BufTable bufs, int kappa,
                                                        int8_t *__restrict__ out, int32_t *__restrict__ expo) {
  const EmuSliceDesc d = descs[blockIdx.x];
  const int line0 = blockIdx.y * 32;
  if (line0 >= d.lines) return;
  const double *src = bufs.p[d.src >> 48] + (d.src & REF_MASK);
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const bool along_lines = d.linestride == 1;
  __shared__ double red[8][33];
  __shared__ int e_line[32];
  __shared__ int8_t dig[EMU_MAX_KAPPA][32][36];     // [slice][line][k in tile], padded rows
  // pass 1: max |a| per line
  double mx = 0.0;
  if (along_lines) {
    const int line = line0 + tx;
    if (line < d.lines)
      for (int a = 0; a < d.n_members; ++a)
        for (int l = ty; l < d.dl; l += 8) mx = fmax(mx, fabs(src[a * d.mstride + l * d.lstride + line]));
    red[ty][tx] = mx;
  } else {
    for (int li = ty; li < 32; li += 8) {
      const int line = line0 + li;
      double m2 = 0.0;
      if (line < d.lines)
        for (int a = 0; a < d.n_members; ++a)
          for (int l = tx; l < d.dl; l += 32) m2 = fmax(m2, fabs(src[a * d.mstride + l * d.lstride + line * d.linestride]));
      for (int o = 16; o > 0; o >>= 1) m2 = fmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
      if (tx == 0) red[0][li] = m2;
    }
  }
  __syncthreads();
  if (threadIdx.x < 32) {
    double m2 = red[0][threadIdx.x];
    if (along_lines) for (int j = 1; j < 8; ++j) m2 = fmax(m2, red[j][threadIdx.x]);
    int e = 0;
    if (m2 > 0.0) frexp(m2, &e);
    e_line[threadIdx.x] = e;
    if (line0 + threadIdx.x < d.lines) expo[d.exp_off + line0 + threadIdx.x] = e;
  }
  __syncthreads();
  // pass 2: digits, 32 lines x 32 k per tile
  const int base_sh = 8 * kappa - 2;
  for (int a = 0; a < d.n_members; ++a)
    for (int l0 = 0; l0 < d.dlpad; l0 += 32) {
      for (int j = 0; j < 4; ++j) {
        int li, l;
        if (along_lines) { li = tx; l = l0 + ty + 8 * j; } else { li = ty + 8 * j; l = l0 + tx; }
        const int line = line0 + li;
        double x = 0.0;
        if (line < d.lines && l < d.dl) x = src[a * d.mstride + l * d.lstride + line * d.linestride];
        int8_t dd[EMU_MAX_KAPPA];
        emu_digits(x, base_sh - e_line[li], kappa, dd);
        for (int s = 0; s < kappa; ++s) dig[s][li][l - l0] = dd[s];
      }
      __syncthreads();
      // 32 lines x 32 bytes per slice: thread t writes the 4-byte word (line t / 8, word t % 8)
      const int li = threadIdx.x >> 3, w = threadIdx.x & 7;
      if (line0 + li < d.lines)
        for (int s = 0; s < kappa; ++s) {
          const int32_t v = *reinterpret_cast<const int32_t *>(&dig[s][li][4 * w]);
          *reinterpret_cast<int32_t *>(out + d.out_off + s * d.plane + (int64_t)(line0 + li) * d.ld + (int64_t)a * d.dlpad + l0 + 4 * w) = v;
        }
      __syncthreads();
    }
}

// Segmented emulated GEMM: one CTA per output tile (128 rows x 64 columns of a psi' block or of one of its
// split-K partial slots); for every segment the kappa anti-diagonal INT32 accumulators are filled by tcgen05
// MMAs and folded into FP64 registers with that segment's exponents and geometry factor.
template <int KAPPA>
__global__ void __launch_bounds__(128) k_emu_stage2(const EmuJob *__restrict__ jobs, const EmuSeg *__restrict__ segs,
                                                    const EmuTile *__restrict__ tiles, BufTable bufs,
                                                    const int8_t *__restrict__ slL, const int8_t *__restrict__ slT,
                                                    const int32_t *__restrict__ exL, const int32_t *__restrict__ exT) {
  constexpr int A_SLICE = 2 * EMU_BM * 16, B_SLICE = 2 * EMU_BN * 16, STAGE = KAPPA * (A_SLICE + B_SLICE);
  constexpr int N_PROD = 96, COPIES = KAPPA * 2 * (EMU_BM + EMU_BN);
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ __align__(8) uint64_t bar_full[EMU_STAGES], bar_empty[EMU_STAGES], bar_done;
  __shared__ uint32_t tmem_slot;
  const EmuTile tl = tiles[blockIdx.x];
  const EmuJob jb = jobs[tl.job];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int m0 = tl.m0, n0 = tl.n0;
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
  uint32_t full_phase = 0, empty_phase = 0, done_phase = 0;
  int use = 0;

  for (int sgi = jb.seg_begin; sgi < jb.seg_end; ++sgi) {
    const EmuSeg sg = segs[sgi];
    const int nsteps = sg.ksteps;
    if (warp == 0) {
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
            for (int t = 0; s + t < KAPPA; ++t)
              umma_i8(tmem + (uint32_t)((s + t) * EMU_BN), da + (uint64_t)((s * A_SLICE) >> 4),
                      db + (uint64_t)((t * B_SLICE) >> 4), idesc, !(k == 0 && s == 0));
          umma_commit(&bar_empty[st]);
        }
        umma_commit(&bar_done);
      }
      __syncwarp();
    } else {
      const int p = tid - 32;
      const int8_t *ga = slL + sg.a_off + (int64_t)m0 * sg.a_ld, *gb = slT + sg.b_off + (int64_t)n0 * sg.b_ld;
      for (int k = 0; k < nsteps + 2; ++k) {
        if (k < nsteps) {
          const int st = (use + k) % EMU_STAGES;
          if (use + k >= EMU_STAGES) { mbar_wait(&bar_empty[st], (empty_phase >> st) & 1u); empty_phase ^= 1u << st; }
          const uint32_t sa = smem_base + st * STAGE, sb = sa + KAPPA * A_SLICE;
          const int64_t kbyte = (int64_t)k * EMU_KS;
          for (int i = p; i < COPIES; i += N_PROD) {
            if (i < KAPPA * 2 * EMU_BM) {
              const int r = i % EMU_BM, c = (i / EMU_BM) & 1, s = i / (2 * EMU_BM);
              const int8_t *g = ga + s * sg.a_plane + (int64_t)r * sg.a_ld + kbyte + c * 16;
              asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa + s * A_SLICE + (c * EMU_BM + r) * 16), "l"(g));
            } else {
              const int i2 = i - KAPPA * 2 * EMU_BM;
              const int r = i2 % EMU_BN, c = (i2 / EMU_BN) & 1, s = i2 / (2 * EMU_BN);
              const int8_t *g = gb + s * sg.b_plane + (int64_t)r * sg.b_ld + kbyte + c * 16;
              asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sb + s * B_SLICE + (c * EMU_BN + r) * 16), "l"(g));
            }
          }
        }
        cp_async_commit();
        if (k >= 2) {
          cp_async_wait<2>();
          asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
          mbar_arrive(&bar_full[(use + k - 2) % EMU_STAGES]);
        }
      }
    }
    use += nsteps;
    mbar_wait(&bar_done, done_phase); done_phase ^= 1u;
    asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
    const int e_row = row < jb.M ? __ldg(exL + sg.ea_off + row) : 0;
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
        const int eb_col = col < jb.N ? __ldg(exT + sg.eb_off + col) : 0;
        facc[c0 + e] += sg.alpha * scalbn(v[e], e_row + eb_col - 2 * (8 * KAPPA - 2));
      }
    }
    asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
    __syncthreads();
  }
  if (row < jb.M) {
    double *C = bufs.p[jb.c >> 48] + (jb.c & REF_MASK);
#pragma unroll
    for (int j = 0; j < EMU_BN; ++j)
      if (n0 + j < jb.N) C[(int64_t)row * jb.c_ld + n0 + j] = facc[j];
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 512);
}

}  // namespace dmrg
