// 3xTF32 contraction engine (DMRG_PREC_TF32X3; "reduced precision in the early sweeps", SURVEY.md
// section 8(a) rows a4-a6 third mode, reading s15): every FP64 value x is split into two TF32 numbers,
// hi = tf32(x) and lo = tf32(x - hi); a product keeps hi*hi + hi*lo + lo*hi (lo*lo ~ 2^-22 is dropped) and is
// accumulated in FP32 in TMEM by tcgen05.mma.kind::tf32.  Tolerance of the mode: 1e-5 relative Frobenius.
// Values must lie inside the FP32 range (the synthetic and chemical inputs here do; no per-line scaling).
//
// The engine reuses the descriptors and the pipeline of emu_seg.cuh: operands are pre-tiled in the shared
// memory layout, one stage = 32 k of both parts, 8 bytes per element in total:
//   A (R = 128): [line tile][k step 32][part (hi, lo)][16-byte chunk (8)][128 rows][4 tf32]
//   B (R = 64):  [line tile][k step 32][16-byte chunk (8)][part (hi, lo)][64 rows][4 tf32]   (hi and lo rows stacked along N)
// A k sub-step of 8 is two MMAs: A_hi x [B_hi | B_lo] (128 x 128 x 8) and A_lo x B_hi (128 x 64 x 8), into TWO FP32
// accumulators (columns 0-63 = hi*hi, 64-127 = hi*lo + lo*hi) that the epilogue adds in FP64; the pair is double
// buffered (256 TMEM columns) so that the drain of a segment overlaps the MMAs of the next.
#pragma once
#include "emu_seg.cuh"

namespace dmrg {

constexpr int TF32_STAGES = 3;
constexpr int TF32_A_PART = 8 * EMU_BM * 16, TF32_B_PART = 8 * EMU_BN * 16;      // bytes of one part of one stage
constexpr int TF32_STAGE = 2 * (TF32_A_PART + TF32_B_PART);

__host__ __device__ constexpr uint32_t umma_idesc_tf32(int M, int N) {           // D = F32, A = B = TF32, K-major, dense
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, bool acc) {
  asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n"
               " tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}\n"
               ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"((uint32_t)acc) : "memory");
}
// x = hi + lo + O(2^-22 |x|), both representable in TF32 (10 explicit mantissa bits): round to nearest by adding
// half an ulp of the dropped 13 bits before masking them
__device__ __forceinline__ void tf32_split(double x, uint32_t &hi, uint32_t &lo) {
  const uint32_t h = (__float_as_uint((float)x) + 0x1000u) & 0xffffe000u;
  const float r = (float)(x - (double)__uint_as_float(h));
  hi = h;
  lo = (__float_as_uint(r) + 0x1000u) & 0xffffe000u;
}

// Full-tile TF32 kernel for dmrg_measure_peak: one CTA per SM, two 128 x 256 FP32 accumulators, back-to-back
// 128 x 256 x 8 MMAs on constant operands (A = 1, B = 0.5: every output of the first accumulator is 4 per MMA).
__global__ void __launch_bounds__(128) k_peak_tf32(int n_mma, float *out) {
  constexpr int M = 128, N = 256;
  __shared__ __align__(128) float sA[2 * M * 4];
  __shared__ __align__(128) float sB[2 * N * 4];
  __shared__ __align__(8) uint64_t bar;
  __shared__ uint32_t tmem_slot;
  const int tid = threadIdx.x, warp = tid >> 5;
  for (int i = tid; i < 2 * M * 4; i += 128) sA[i] = 1.0f;
  for (int i = tid; i < 2 * N * 4; i += 128) sB[i] = 0.5f;
  if (warp == 0) tmem_alloc(&tmem_slot, 512);
  if (tid == 0) mbar_init(&bar, 1);
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const uint32_t tmem = tmem_slot;
  if (tid == 0) {
    const uint64_t ad = umma_smem_desc((uint32_t)__cvta_generic_to_shared(sA), M * 16, 128);
    const uint64_t bd = umma_smem_desc((uint32_t)__cvta_generic_to_shared(sB), N * 16, 128);
    const uint32_t idesc = umma_idesc_tf32(M, N);
    for (int j = 0; j < n_mma; ++j) umma_tf32(tmem + (uint32_t)((j & 1) * 256), ad, bd, idesc, j >= 2);
    umma_commit(&bar);
  }
  mbar_wait(&bar, 0);
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  if (out != nullptr && blockIdx.x == 0) {
    int32_t v[8];
    tmem_ld8(tmem + ((uint32_t)(warp * 32) << 16), v);
    out[tid] = __int_as_float(v[0]);
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 512);
}

// Split-and-pack, same descriptors as k_emu_slice_desc (exponent fields unused).  grid = (descriptors, 64-line
// groups), 256 threads.  linestride == 1: thread = (line, 8 consecutive k) and writes two 16-byte chunks per part,
// consecutive lanes = consecutive lines = consecutive chunks; lstride == 1: thread = (8 lines, one k).
__global__ void __launch_bounds__(256) k_tf32_slice_desc(const EmuSliceDesc *__restrict__ descs, const int2 *__restrict__ work, BufTable bufs,
                                                         unsigned char *__restrict__ out) {
  const int2 wk = work[blockIdx.x];                  // (descriptor, first line of the 64-line tile): one CTA per tile that exists
  const EmuSliceDesc d = descs[wk.x];
  const int line0 = wk.y;
  if (line0 >= d.lines || d.bound == 2) return;      // bound == 2: written by the stage-1 epilogue
  const double *src = bufs.p[d.src >> 48] + (d.src & REF_MASK);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int R = (int)d.tile_rows, ksteps = (int)(d.ld >> 5);
  const bool along_lines = d.linestride == 1;
  const int lx = tid & 63, ky = tid >> 6;
  for (int ks = 0; ks < ksteps; ++ks) {
    if (along_lines) {
      const int line = line0 + lx;
      if (line >= d.lines) continue;
      const int gl = d.line_base + line;
      // 128-row units are group-major, [8-row group][part][chunk][8 rows][16 B] (a ragged tile of k_tf32_seg loads only the
      // groups that exist, as in k_emu_seg); 64-row units [chunk][part][row] (hi and lo rows stacked along N)
      const int row = gl % R;
      unsigned char *stage = out + (d.out_off + ((int64_t)(gl / R) * ksteps + ks) * (R * 32)) * 8 +
                             (R == 128 ? (row >> 3) * 2048 + (row & 7) * 16 : row * 16);
      int a = ((ks << 5) + ky * 8) / d.dlpad, l = (ks << 5) + ky * 8 - a * d.dlpad;
      uint32_t hi[8], lo[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const double x = (a < d.n_members && l < d.dl) ? src[a * d.mstride + l * d.lstride + line] : 0.0;
        tf32_split(x, hi[j], lo[j]);
        if (++l == d.dlpad) { l = 0; ++a; }
      }
#pragma unroll
      for (int c = 0; c < 2; ++c) {                   // chunk ky * 2 + c of both parts
        unsigned char *p = stage + (ky * 2 + c) * (R == 128 ? 128 : 2 * R * 16);
        *reinterpret_cast<uint4 *>(p) = make_uint4(hi[4 * c], hi[4 * c + 1], hi[4 * c + 2], hi[4 * c + 3]);
        *reinterpret_cast<uint4 *>(p + (R == 128 ? 1024 : R * 16)) = make_uint4(lo[4 * c], lo[4 * c + 1], lo[4 * c + 2], lo[4 * c + 3]);
      }
    } else {
      const int k = (ks << 5) + lane, a = k / d.dlpad, l = k - a * d.dlpad;
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int line = line0 + warp * 8 + j;
        if (line >= d.lines) continue;
        const int gl = d.line_base + line;
        const double x = (a < d.n_members && l < d.dl) ? src[a * d.mstride + l * d.lstride + line * d.linestride] : 0.0;
        uint32_t hi, lo;
        tf32_split(x, hi, lo);
        const int row = gl % R;
        unsigned char *p = out + (d.out_off + ((int64_t)(gl / R) * ksteps + ks) * (R * 32)) * 8 + (lane & 3) * 4 +
                           (R == 128 ? (row >> 3) * 2048 + (lane >> 2) * 128 + (row & 7) * 16 : (lane >> 2) * (2 * R * 16) + row * 16);
        *reinterpret_cast<uint32_t *>(p) = hi;
        *reinterpret_cast<uint32_t *>(p + (R == 128 ? 1024 : R * 16)) = lo;
      }
    }
  }
}

// 16 epilogue warps of 16 columns (the FP32 epilogue needs 96 registers per thread, so twice the warps of k_emu_seg fit;
// measured 5 % faster at configs[2]); warp 0 = MMA issuer, warp 1 = producer as in k_emu_seg
constexpr int TF32_EPI_WARPS = 16;
constexpr int TF32_THREADS = 64 + 32 * TF32_EPI_WARPS;
__device__ __forceinline__ void tf32_epi_bar() {
  asm volatile("bar.sync 1, %0;\n" ::"n"(32 * TF32_EPI_WARPS) : "memory");
}
// Segmented 3xTF32 GEMM: the roles, barriers and tile schedule of k_emu_seg.  TMEM holds two accumulator pairs
// (columns 0-127 and 128-255); segment i uses pair i & 1, `tfree[b]` returns a pair to the MMA warp.
__global__ void __launch_bounds__(TF32_THREADS, 1) k_tf32_seg(const EmuJob *__restrict__ jobs, const EmuSeg *__restrict__ segs,
                                                             const EmuTile *__restrict__ tiles, const int *__restrict__ cta_begin,
                                                             BufTable bufs, const unsigned char *__restrict__ slA,
                                                             const unsigned char *__restrict__ slB,
                                                             unsigned char *__restrict__ fuse_out,
                                                             int *__restrict__ gang, int epoch) {
  extern __shared__ __align__(128) unsigned char smem[];     // TF32_STAGES stages, then the 128 x 33 transpose tile
  __shared__ __align__(8) uint64_t bar_full[TF32_STAGES], bar_empty[TF32_STAGES], bar_done[2], bar_tfree[2];
  __shared__ uint32_t tmem_slot;
  __shared__ int64_t s_coff[EMU_BN];
  __shared__ double s_scale[EMU_BN];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t smem_base = (uint32_t)__cvta_generic_to_shared(smem);

  if (warp == 0) tmem_alloc(&tmem_slot, 256);
  if (tid == 0) {
    for (int s = 0; s < TF32_STAGES; ++s) { mbar_init(&bar_full[s], 1); mbar_init(&bar_empty[s], 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(&bar_done[b], 1); mbar_init(&bar_tfree[b], TF32_EPI_WARPS); }
  }
  asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const uint32_t tmem = tmem_slot;
  const int t_begin = cta_begin[blockIdx.x], t_end = cta_begin[blockIdx.x + 1];

  if (warp == 0) {
    // ---------------------------------------------------------------- MMA issuer (all lanes walk the lists, one issues:
    // tc_i8.cuh elect_one)
    {
      const bool leader = elect_one();
      const uint32_t idesc = umma_idesc_tf32(EMU_BM, EMU_BN), idesc2 = umma_idesc_tf32(EMU_BM, 2 * EMU_BN);
      uint32_t full_phase = 0, tfree_phase = 0;
      int use = 0, item = 0;
      for (int t = t_begin; t < t_end; ++t) {
        const EmuJob jb = jobs[tiles[t].job];
        for (int sgi = jb.seg_begin; sgi < jb.seg_end; ++sgi, ++item) {
          const int nsteps = segs[sgi].ksteps, buf = item & 1;
          if (item >= 2) { mbar_wait(&bar_tfree[buf], (tfree_phase >> buf) & 1u); tfree_phase ^= 1u << buf; }
          asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
          for (int k = 0; k < nsteps; ++k) {
            const int st = (use + k) % TF32_STAGES;
            mbar_wait(&bar_full[st], (full_phase >> st) & 1u); full_phase ^= 1u << st;
            asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
            const uint32_t sa = smem_base + st * TF32_STAGE, sb = sa + 2 * TF32_A_PART;
#pragma unroll
            for (int j = 0; j < 4; ++j) {             // four k sub-steps of 8 (two 16-byte chunks each)
              // A: [8-row group][part][chunk][8 rows][16 B]: chunks 128 B apart, row groups 2 KB apart, lo part at + 1 KB
              const uint64_t ah = umma_smem_desc(sa + j * 256, 128, 2048);
              const uint64_t al = umma_smem_desc(sa + 1024 + j * 256, 128, 2048);
              // rows 0-63 of a B chunk = hi part, rows 64-127 = lo part: one descriptor serves N = 64 (hi) and N = 128 (hi | lo)
              const uint64_t bs = umma_smem_desc(sb + j * 2 * (2 * EMU_BN * 16), 2 * EMU_BN * 16, 128);
              const uint32_t dcol = tmem + (uint32_t)(buf * 2 * EMU_BN);
              // two accumulators: columns 0-63 = hi*hi, columns 64-127 = hi*lo + lo*hi (summed in FP64 by the epilogue)
              if (leader) {
                umma_tf32(dcol, ah, bs, idesc2, !(k == 0 && j == 0));   // A_hi x [B_hi | B_lo], N = 128
                umma_tf32(dcol + EMU_BN, al, bs, idesc, true);          // A_lo x B_hi, N = 64
              }
            }
            if (leader) umma_commit(&bar_empty[st]);
            __syncwarp();
          }
          if (leader) umma_commit(&bar_done[buf]);
          __syncwarp();
          use += nsteps;
        }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ---------------------------------------------------------------- producer
    if (lane == 0) {
      uint32_t empty_phase = 0;
      int use = 0;
      for (int t = t_begin; t < t_end; ++t) {
        const EmuTile tl = tiles[t];
        const EmuJob jb = jobs[tl.job];
        GangSync gs(gang, tl, jb, epoch);     // see emu_seg.cuh
        const int rowsA = jb.fuse ? EMU_BM : min(EMU_BM, (jb.M - tl.m0 + 7) & ~7);
        const uint32_t a_bytes = (uint32_t)(rowsA >> 3) * 2048;
        for (int sgi = jb.seg_begin; sgi < jb.seg_end; ++sgi) {
          gs.arrive(sgi - jb.seg_begin);
          const EmuSeg sg = segs[sgi];
          const unsigned char *ga = slA + (sg.a_off + (int64_t)(tl.m0 / EMU_BM) * sg.ksteps * (EMU_BM * 32)) * 8;
          const unsigned char *gb = slB + (sg.b_off + (int64_t)(tl.n0 / EMU_BN) * sg.ksteps * (EMU_BN * 32)) * 8;
          for (int k = 0; k < sg.ksteps; ++k) {
            const int st = (use + k) % TF32_STAGES;
            if (use + k >= TF32_STAGES) { mbar_wait(&bar_empty[st], (empty_phase >> st) & 1u); empty_phase ^= 1u << st; }
            const uint32_t sa = smem_base + st * TF32_STAGE, sb = sa + 2 * TF32_A_PART;
            mbar_expect_tx(&bar_full[st], a_bytes + 2 * TF32_B_PART);
            bulk_g2s(sa, ga + (int64_t)k * (2 * TF32_A_PART), a_bytes, &bar_full[st]);   // the row groups of the tile that exist
            bulk_g2s(sb, gb + (int64_t)k * (2 * TF32_B_PART), 2 * TF32_B_PART, &bar_full[st]);
          }
          use += sg.ksteps;
        }
      }
    }
    __syncwarp();
  } else {
    // ---------------------------------------------------------------- epilogue
    const int ew = warp - 2, etid = tid - 64;
    const int quarter = warp & 3, cgrp = ew >> 2, trow = quarter * 32 + lane;
    constexpr int CPW = EMU_BN / (TF32_EPI_WARPS / 4);
    double(*xpose)[33] = reinterpret_cast<double(*)[33]>(smem + TF32_STAGES * TF32_STAGE);
    uint32_t done_phase = 0;
    int item = 0;
    for (int t = t_begin; t < t_end; ++t) {
      const EmuTile tl = tiles[t];
      const EmuJob jb = jobs[tl.job];
      const int m0 = tl.m0, n0 = tl.n0, row = m0 + trow;
      int64_t roff = 0;
      double rscale = 1.0;
      int r_hi = 0, r_lo = 0;
      if (jb.rows_split) {
        const int hi = row / jb.n1, lo = row - hi * jb.n1;
        r_hi = hi; r_lo = lo;
        roff = lo + hi * jb.c_nhi;
        if (jb.scale >= 0 && row < jb.M) rscale = (bufs.p[jb.scale >> 48] + (jb.scale & REF_MASK))[hi];
      } else if (etid < EMU_BN) {
        const int n = n0 + etid, hi = n / jb.n1, lo = n - hi * jb.n1;
        s_coff[etid] = lo + hi * jb.c_nhi;
        s_scale[etid] = (jb.scale >= 0 && n < jb.N) ? (bufs.p[jb.scale >> 48] + (jb.scale & REF_MASK))[hi] : 1.0;
      }
      double facc[CPW];
#pragma unroll
      for (int j = 0; j < CPW; ++j) facc[j] = 0.0;
      for (int sgi = jb.seg_begin; sgi < jb.seg_end; ++sgi, ++item) {
        const double alpha = segs[sgi].alpha;
        const int buf = item & 1;
        mbar_wait(&bar_done[buf], (done_phase >> buf) & 1u); done_phase ^= 1u << buf;
        asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
        const uint32_t tbase = tmem + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(buf * 2 * EMU_BN + cgrp * CPW);
        int32_t pv[CPW / 8][8], ps[CPW / 8][8];
#pragma unroll
        for (int g8 = 0; g8 < CPW / 8; ++g8) {
          tmem_ld8_nowait(tbase + (uint32_t)(g8 * 8), pv[g8]);
          tmem_ld8_nowait(tbase + (uint32_t)(EMU_BN + g8 * 8), ps[g8]);
        }
        tmem_ld_wait();
        asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(&bar_tfree[buf]);
#pragma unroll
        for (int g8 = 0; g8 < CPW / 8; ++g8)
#pragma unroll
          for (int e = 0; e < 8; ++e)
            facc[g8 * 8 + e] = fma((double)__int_as_float(pv[g8][e]) + (double)__int_as_float(ps[g8][e]), alpha, facc[g8 * 8 + e]);
      }
      double *C = bufs.p[jb.c >> 48] + (jb.c & REF_MASK);
      if (jb.rows_split) {
        if (row < jb.M && (!jb.fuse || jb.write_fp64)) {
#pragma unroll
          for (int j = 0; j < CPW; ++j) {
            const int col = n0 + cgrp * CPW + j;
            if (col < jb.N) C[roff + (int64_t)col * jb.c_ld] = facc[j] * rscale;
          }
        }
        if (row < jb.M && jb.fuse) {
          // hi / lo parts of T for stage 2, straight from the accumulators (see k_emu_seg): four consecutive l of
          // line r' = one 16-byte chunk per part; consecutive lanes = consecutive lines = consecutive chunks
          const int pc = r_hi / jb.per_piece, a_loc = r_hi - pc * jb.per_piece;
          const int ksteps_pc = (pc == jb.n_pieces - 1 ? jb.ld_last : jb.ld_full) >> 5;
          unsigned char *unit = fuse_out + (jb.t_out_off + (int64_t)pc * jb.piece_bytes + (int64_t)(r_lo >> 6) * ksteps_pc * (EMU_BN * 32)) * 8 +
                                (r_lo & 63) * 16;
#pragma unroll
          for (int q4 = 0; q4 < CPW / 4; ++q4) {
            const int l0 = n0 + cgrp * CPW + q4 * 4;
            if (l0 >= jb.dlpad) continue;
            uint32_t hi[4], lo[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) tf32_split(l0 + j < jb.N ? facc[q4 * 4 + j] * rscale : 0.0, hi[j], lo[j]);
            const int k = a_loc * jb.dlpad + l0;
            unsigned char *dst = unit + (int64_t)(k >> 5) * (2 * TF32_B_PART) + ((k & 31) >> 2) * (2 * EMU_BN * 16);
            *reinterpret_cast<uint4 *>(dst) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
            *reinterpret_cast<uint4 *>(dst + EMU_BN * 16) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
            if (l0 + 4 == jb.dlpad) {             // zero the 16 elements that pad the unit's K to a multiple of 32
              const int members = jb.M / jb.n1;
              const int na = pc == jb.n_pieces - 1 ? members - pc * jb.per_piece : jb.per_piece;
              if (a_loc == na - 1 && ((na * jb.dlpad) & 31) == 16) {
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                  const int k2 = na * jb.dlpad + 4 * i;
                  unsigned char *d2 = unit + (int64_t)(k2 >> 5) * (2 * TF32_B_PART) + ((k2 & 31) >> 2) * (2 * EMU_BN * 16);
                  *reinterpret_cast<uint4 *>(d2) = make_uint4(0u, 0u, 0u, 0u);
                  *reinterpret_cast<uint4 *>(d2 + EMU_BN * 16) = make_uint4(0u, 0u, 0u, 0u);
                }
              }
            }
          }
        }
        continue;
      }
      tf32_epi_bar();                                  // s_coff / s_scale visible
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        if (cgrp * CPW / 32 == h) {
#pragma unroll
          for (int j = 0; j < CPW; ++j) xpose[trow][(cgrp * CPW) % 32 + j] = facc[j];
        }
        tf32_epi_bar();
        const int col = h * 32 + lane;
        if (n0 + col < jb.N) {
          const double sc = s_scale[col];
          const int64_t co = s_coff[col];
          for (int r = ew; r < EMU_BM && m0 + r < jb.M; r += TF32_EPI_WARPS) C[(int64_t)(m0 + r) * jb.c_ld + co] = xpose[r][lane] * sc;
        }
        tf32_epi_bar();
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 256);
}

}  // namespace dmrg
