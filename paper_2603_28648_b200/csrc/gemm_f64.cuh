// k_gemm_f64: the generic, output-stationary grouped GEMM that executes every descriptor list
// of plan.cpp (H_eff stage 1 / stage 2, rotation, integral contraction) in native FP64:
//     C[m][n] = colscale[n / n1] * sum_seg alpha_seg * sum_k A_seg[m][k] B_seg[k][n]
// tcgen05 has no FP64 kind on sm_100a (ptxas rejects .kind::f64), so the FP64 tensor path is
// warp-level mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4).  The DMMA pipe issues one instruction per
// ~20 clocks per SM sub-partition, so the kernel spends few issue slots around each DMMA:
// operands go global -> shared with cp.async (LDGSTS, no register staging) through a 3-stage
// ring; addressing is set up once per segment and advanced by additions; full K blocks take a
// predicate-free fast path; shared-memory tiles are padded so that fragment loads and the
// cp.async stores are bank-conflict free; the MMA block exists in compile-time layout variants.
// Each CTA owns one output tile and walks that tile's segment list, accumulating in registers:
// no atomics, deterministic, one write per output element.
#pragma once
#include <cuda_runtime.h>

#include "backend.h"

namespace dmrg {

static constexpr int64_t REF_MASK = (1LL << 48) - 1;
static constexpr int FLAT_IDX = 1 << 30;

__device__ __forceinline__ const double *rd_ref(const BufTable &b, ref_t r) {
  return b.p[r >> 48] + (r & REF_MASK);
}
__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
// 8-byte copy, issued only when `on` (a predicated instruction, no branch)
__device__ __forceinline__ void cp_async8(uint32_t dst, const double *src, bool on) {
  asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %2, 0;\n @p cp.async.ca.shared.global [%0], [%1], 8;\n}\n"
               ::"r"(dst), "l"(src), "r"((int)on));
}
// same, zero-filling the destination when `valid` is false (src must still be a mapped address)
__device__ __forceinline__ void cp_async8_zfill(uint32_t dst, const double *src, bool on, bool valid) {
  asm volatile("{\n .reg .pred p;\n setp.ne.b32 p, %3, 0;\n @p cp.async.ca.shared.global [%0], [%1], 8, %2;\n}\n"
               ::"r"(dst), "l"(src), "r"(valid ? 8 : 0), "r"((int)on));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

template <int MT> struct GemmCfg {
  static constexpr int BM = 16 * MT, BN = 16 * MT, BK = 16, NSTAGE = 3, THREADS = 128;
  static constexpr int E = 2 * MT;   // 8-byte elements per thread per operand tile
  // layout 0: [row][k] with row stride BK + 4; layout 1: [k][row] with row stride BM + 4
  static constexpr int LD0 = BK + 4, LD1 = BM + 4;
  static constexpr int TILE_ELEMS = (BM * LD0 > BK * LD1) ? BM * LD0 : BK * LD1;
  static constexpr int MAX_STRIP = 8;   // n-tiles per CTA (plan.cpp STRIP)
  static constexpr int SMEM_BYTES = NSTAGE * 2 * TILE_ELEMS * 8 + NSTAGE * 16 + MAX_STRIP * BN * 8;
};

// One 16-deep K block on the tensor pipe.  LA / LB are the shared-memory layouts of the tiles.
// Rows / columns beyond the matrix edge hold stale data; they only reach accumulators that the
// epilogue never stores.
template <int MT, int LA, int LB>
__device__ __forceinline__ void mma_block(double (&acc)[MT][MT][2], const double *as, const double *bs, int wm,
                                          int wn, int lane, double alpha) {
  using G = GemmCfg<MT>;
  const int r = lane >> 2, c = lane & 3;
  const double *pa = LA == 0 ? as + (wm * 8 * MT + r) * G::LD0 + c : as + c * G::LD1 + wm * 8 * MT + r;
  const double *pb = LB == 0 ? bs + (wn * 8 * MT + r) * G::LD0 + c : bs + c * G::LD1 + wn * 8 * MT + r;
#pragma unroll
  for (int ks = 0; ks < G::BK / 4; ++ks) {
    double af[MT], bf[MT];
#pragma unroll
    for (int i = 0; i < MT; ++i) af[i] = (LA == 0 ? pa[i * 8 * G::LD0 + ks * 4] : pa[ks * 4 * G::LD1 + i * 8]);
#pragma unroll
    for (int j = 0; j < MT; ++j)
      bf[j] = alpha * (LB == 0 ? pb[j * 8 * G::LD0 + ks * 4] : pb[ks * 4 * G::LD1 + j * 8]);
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
      for (int j = 0; j < MT; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
  }
}

// ROLE only names the instantiation (profiles list the launches by role): 0 integral contraction (a3),
// 1 rotation stage 1, 2 rotation stage 2 (a9), 3 H_eff stage 1 (a5), 4 H_eff stage 2 (a6).
//
// Global -> shared thread mappings (t15 = tid % 16, t4 = tid / 16, element j < 2 MT):
//   layout 0 (k is the unit-stride index): k = t15, row = t4 + 8 j
//   layout 1 (row is the unit-stride index): row = t15 + 16 (j % MT), k = t4 + 8 (j / MT)
// so that a half-warp always copies 16 consecutive doubles into 16 distinct banks.
template <int MT, int ROLE>
__global__ void __launch_bounds__(128) k_gemm_f64(const JobDesc *__restrict__ jobs,
                                                  const SegDesc *__restrict__ segs,
                                                  const TileDesc *__restrict__ tiles,
                                                  const __grid_constant__ BufTable bufs) {
  using G = GemmCfg<MT>;
  constexpr int BK = G::BK, BN = G::BN, E = G::E, NS = G::NSTAGE, LD0 = G::LD0, LD1 = G::LD1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double *As = reinterpret_cast<double *>(smem_raw);
  double *Bs = As + NS * G::TILE_ELEMS;
  double *meta = Bs + NS * G::TILE_ELEMS;        // per stage: alpha, layout flags (as a double)
  int2 *coltab = reinterpret_cast<int2 *>(meta + NS * 2);   // (n / n1, n % n1) of every column of the strip

  const TileDesc td = tiles[blockIdx.x];
  const JobDesc jd = jobs[td.job];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, wm = warp & 1, wn = warp >> 1;
  const int t15 = tid & 15, t4 = tid >> 4;
  const int m0 = td.m0;
  const int Mrem = jd.M - m0;                     // > 0
  const int n1 = jd.n1;
  const int strip = td.work;                      // consecutive n-tiles handled by this CTA (>= 1)

  double acc[MT][MT][2];
#pragma unroll
  for (int i = 0; i < MT; ++i)
#pragma unroll
    for (int j = 0; j < MT; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  // ---- producer state: set up once per segment, advanced by additions per K block
  int pseg = jd.seg_begin, pk0 = 0, pK = 0, p_n0 = td.n0, p_left = strip;
  const int seg_end = jd.seg_end;
  const double *a_row = nullptr, *pA = nullptr, *pB = nullptr;
  int64_t boff[E];                                 // per-column offsets of this thread's B elements
  int64_t a_khi = 0, a_jstep = 0, a_kstep = 0, b_kstep = 0;
  int a_kq = 0, a_kr = 0, a_q16 = 0, a_r16 = 0, a_kn1 = FLAT_IDX, a_klo = 0, p_la = 0, p_lb = 0;
  uint32_t amask = 0, bmask = 0;                   // bit j: element j lies inside the matrix
  double p_alpha = 1.0;
  const uint32_t smem_a = (uint32_t)__cvta_generic_to_shared(As), smem_b = (uint32_t)__cvta_generic_to_shared(Bs);
  // shared-memory byte offsets of element 0 under both layouts (the same for A and B: BM == BN)
  const uint32_t dst0 = (uint32_t)(t4 * LD0 + t15) * 8u, dst1 = (uint32_t)(t4 * LD1 + t15) * 8u;

  auto setup_segment = [&]() {
    const SegDesc sd = segs[pseg];
    const int Nrem = jd.N - p_n0;
    pK = sd.K; pk0 = 0; p_alpha = sd.alpha;
    const double *Ap = rd_ref(bufs, sd.a), *Bp = rd_ref(bufs, sd.b);
    p_la = (sd.a_ms == 1 && sd.a_klo != 1) ? 1 : 0;
    p_lb = (sd.b_nlo == 1 && sd.b_ks != 1) ? 1 : 0;
    a_kn1 = sd.a_kn1; a_klo = sd.a_klo; a_khi = sd.a_khi;
    amask = bmask = 0;
    if (p_la == 0) {
      a_row = Ap + (int64_t)(m0 + min(t4, Mrem - 1)) * sd.a_ms;
      a_jstep = 8 * (int64_t)sd.a_ms;
      if (a_kn1 == FLAT_IDX) { a_kq = 0; a_kr = t15; a_q16 = 0; a_r16 = BK; }
      else { a_kq = t15 / a_kn1; a_kr = t15 - a_kq * a_kn1; a_q16 = BK / a_kn1; a_r16 = BK - a_q16 * a_kn1; }
#pragma unroll
      for (int j = 0; j < E; ++j) amask |= (t4 + 8 * j < Mrem) ? (1u << j) : 0u;
    } else {                                       // layout 1 is only planned with a flat k index
      pA = Ap + (int64_t)(m0 + min(t15, Mrem - 1)) * sd.a_ms + (int64_t)t4 * sd.a_klo;
      a_jstep = 16 * (int64_t)sd.a_ms;
      a_kstep = 8 * (int64_t)sd.a_klo;
#pragma unroll
      for (int j = 0; j < E; ++j) amask |= (t15 + 16 * (j % MT) < Mrem) ? (1u << j) : 0u;
    }
    b_kstep = 8 * (int64_t)sd.b_ks;
    auto col_off = [&](int nn) -> int64_t {
      const int2 q = coltab[p_n0 - td.n0 + min(nn, Nrem - 1)];   // clamp: out-of-range columns are never copied
      return (int64_t)q.x * sd.b_nhi + (int64_t)q.y * sd.b_nlo;
    };
    if (p_lb == 0) {
      pB = Bp + (int64_t)t15 * sd.b_ks;
#pragma unroll
      for (int j = 0; j < E; ++j) { boff[j] = col_off(t4 + 8 * j); bmask |= (t4 + 8 * j < Nrem) ? (1u << j) : 0u; }
    } else {
      pB = Bp + (int64_t)t4 * sd.b_ks;
#pragma unroll
      for (int c = 0; c < MT; ++c) boff[c] = col_off(t15 + 16 * c);
#pragma unroll
      for (int j = 0; j < E; ++j) bmask |= (t15 + 16 * (j % MT) < Nrem) ? (1u << j) : 0u;
    }
  };

  // Issue the cp.async copies of the next K block into ring slot `stage` (always commits a group).
  // All copies are predicated instructions; there is no branch inside the element loops.
  auto produce = [&](int stage) {
    if (p_left > 0) {
      if (pK == 0) setup_segment();
      const uint32_t sa = smem_a + stage * (G::TILE_ELEMS * 8), sb = smem_b + stage * (G::TILE_ELEMS * 8);
      const int krem = pK - pk0;
      if (krem >= BK) {                            // full K block: no k predicate, no zero fill
        if (p_la == 0) {
          const double *p = a_row + (int64_t)a_kq * a_khi + (int64_t)a_kr * a_klo;
#pragma unroll
          for (int j = 0; j < E; ++j) { cp_async8(sa + dst0 + j * (8 * LD0 * 8), p, (amask >> j) & 1u); p += a_jstep; }
        } else {
#pragma unroll
          for (int j = 0; j < E; ++j)
            cp_async8(sa + dst1 + (uint32_t)((j / MT) * 8 * LD1 + 16 * (j % MT)) * 8u,
                      pA + (j % MT) * a_jstep + (j / MT) * a_kstep, (amask >> j) & 1u);
        }
        if (p_lb == 0) {
#pragma unroll
          for (int j = 0; j < E; ++j) cp_async8(sb + dst0 + j * (8 * LD0 * 8), pB + boff[j], (bmask >> j) & 1u);
        } else {
#pragma unroll
          for (int j = 0; j < E; ++j)
            cp_async8(sb + dst1 + (uint32_t)((j / MT) * 8 * LD1 + 16 * (j % MT)) * 8u,
                      pB + boff[j % MT] + (j / MT) * b_kstep, (bmask >> j) & 1u);
        }
      } else {                                     // ragged tail of a segment: zero-fill k >= krem
        if (p_la == 0) {
          const bool kok = t15 < krem;
          const double *p = a_row + (int64_t)a_kq * a_khi + (int64_t)a_kr * a_klo;
#pragma unroll
          for (int j = 0; j < E; ++j) {
            cp_async8_zfill(sa + dst0 + j * (8 * LD0 * 8), kok ? p : a_row, (amask >> j) & 1u, kok);
            p += a_jstep;
          }
        } else {
#pragma unroll
          for (int j = 0; j < E; ++j) {
            const bool kok = t4 + 8 * (j / MT) < krem;
            cp_async8_zfill(sa + dst1 + (uint32_t)((j / MT) * 8 * LD1 + 16 * (j % MT)) * 8u,
                            kok ? pA + (j % MT) * a_jstep + (j / MT) * a_kstep : pA, (amask >> j) & 1u, kok);
          }
        }
        if (p_lb == 0) {
          const bool kok = t15 < krem;
#pragma unroll
          for (int j = 0; j < E; ++j)
            cp_async8_zfill(sb + dst0 + j * (8 * LD0 * 8), kok ? pB + boff[j] : pB, (bmask >> j) & 1u, kok);
        } else {
#pragma unroll
          for (int j = 0; j < E; ++j) {
            const bool kok = t4 + 8 * (j / MT) < krem;
            cp_async8_zfill(sb + dst1 + (uint32_t)((j / MT) * 8 * LD1 + 16 * (j % MT)) * 8u,
                            kok ? pB + boff[j % MT] + (j / MT) * b_kstep : pB, (bmask >> j) & 1u, kok);
          }
        }
      }
      if (tid == 0) { meta[stage * 2] = p_alpha; meta[stage * 2 + 1] = (double)(p_la * 2 + p_lb); }
      // advance to the next K block / segment / n-tile of the strip
      pk0 += BK;
      if (pk0 >= pK) {
        pk0 = 0; pK = 0;
        if (++pseg == seg_end) { pseg = jd.seg_begin; p_n0 += BN; --p_left; }
      } else {
        pB += 2 * b_kstep;
        if (p_la == 0) { a_kq += a_q16; a_kr += a_r16; if (a_kr >= a_kn1) { a_kr -= a_kn1; ++a_kq; } }
        else pA += 2 * a_kstep;
      }
    }
    cp_async_commit();
  };

  // epilogue of one n-tile: one write per element, optional per-column-group scale
  double *C = const_cast<double *>(rd_ref(bufs, jd.c));
  const double *scale = jd.scale >= 0 ? rd_ref(bufs, jd.scale) : nullptr;
  auto epilogue = [&](int n0, int Nrem) {
#pragma unroll
    for (int j = 0; j < MT; ++j) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int nn = wn * 8 * MT + j * 8 + 2 * (lane & 3) + e;
        if (nn < Nrem) {
          const int2 q = coltab[n0 - td.n0 + nn];
          const int nq = q.x, nr = q.y;
          const double sc = scale ? __ldg(scale + nq) : 1.0;
          double *cp = C + (int64_t)nq * jd.c_nhi + (int64_t)nr * jd.c_nlo;
#pragma unroll
          for (int i = 0; i < MT; ++i) {
            const int mm = wm * 8 * MT + i * 8 + (lane >> 2);
            if (mm < Mrem) cp[(int64_t)(m0 + mm) * jd.c_ms] = acc[i][j][e] * sc;
          }
        }
#pragma unroll
        for (int i = 0; i < MT; ++i) acc[i][j][e] = 0.0;
      }
    }
  };

  const int n_iters = jd.n_iters;         // K blocks per n-tile: sum over segments of ceil(K / 16)
  for (int idx = tid; idx < strip * BN && td.n0 + idx < jd.N; idx += 128) {
    const int n = td.n0 + idx;
    int nq = 0, nr = n;
    if (n1 != FLAT_IDX) { nq = n / n1; nr = n - nq * n1; }
    coltab[idx] = make_int2(nq, nr);
  }
  __syncthreads();
  if (n_iters == 0) {                     // a job without segments writes zeros
    for (int s = 0, n0 = td.n0; s < strip; ++s, n0 += BN) epilogue(n0, jd.N - n0);
    return;
  }
#pragma unroll
  for (int s = 0; s < NS - 1; ++s) produce(s);
  int c_n0 = td.n0, c_it = 0, stage = 0;
  const int total = n_iters * strip;
  for (int it = 0; it < total; ++it) {
    cp_async_wait<NS - 2>();
    __syncthreads();
    produce(stage == 0 ? NS - 1 : stage - 1);
    const int Nrem = jd.N - c_n0;
    if ((wm * 8 * MT < Mrem) && (wn * 8 * MT < Nrem)) {
      const double *as = As + stage * G::TILE_ELEMS, *bs = Bs + stage * G::TILE_ELEMS;
      const double alpha = meta[stage * 2];
      const int lay = (int)meta[stage * 2 + 1];
      switch (lay) {
        case 0: mma_block<MT, 0, 0>(acc, as, bs, wm, wn, lane, alpha); break;
        case 1: mma_block<MT, 0, 1>(acc, as, bs, wm, wn, lane, alpha); break;
        case 2: mma_block<MT, 1, 0>(acc, as, bs, wm, wn, lane, alpha); break;
        default: mma_block<MT, 1, 1>(acc, as, bs, wm, wn, lane, alpha); break;
      }
    }
    if (++c_it == n_iters) { epilogue(c_n0, Nrem); c_it = 0; c_n0 += BN; }
    stage = stage == NS - 1 ? 0 : stage + 1;
  }
  cp_async_wait<0>();
}

}  // namespace dmrg
