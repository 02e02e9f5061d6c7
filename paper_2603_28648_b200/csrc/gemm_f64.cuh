// k_gemm_f64: the generic, output-stationary grouped GEMM that executes every descriptor list
// of plan.cpp (H_eff stage 1 / stage 2, rotation, integral contraction) in native FP64:
//     C[m][n] = colscale[n / n1] * sum_seg alpha_seg * sum_k A_seg[m][k] B_seg[k][n]
// tcgen05 has no FP64 kind on sm_100a (ptxas rejects .kind::f64), so the FP64 tensor path is
// warp-level mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4).  The DMMA pipe issues one instruction per
// ~20 clocks per SM sub-partition, so the kernel is written to spend few issue slots around each
// DMMA: operands go global -> shared with cp.async (LDGSTS, zero-fill predication, no register
// staging) through a 3-stage ring, all addressing is set up once per segment and advanced by
// additions, shared-memory tiles are padded so that fragment loads and the cp.async stores are
// bank-conflict free, and the MMA block exists in four compile-time layout variants.
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
__device__ __forceinline__ void cp_async8(uint32_t dst, const double *src, bool valid) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(valid ? 8 : 0));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

template <int MT> struct GemmCfg {
  static constexpr int BM = 16 * MT, BN = 16 * MT, BK = 16, NSTAGE = 3, THREADS = 128;
  static constexpr int EA = BM * BK / THREADS, EB = BK * BN / THREADS;
  // layout 0: [row][k] with row stride BK + 4; layout 1: [k][row] with row stride BM + 4
  static constexpr int LD0 = BK + 4, LD1 = BM + 4;
  static constexpr int TILE_ELEMS = (BM * LD0 > BK * LD1) ? BM * LD0 : BK * LD1;
  static constexpr int SMEM_BYTES = NSTAGE * 2 * TILE_ELEMS * 8 + NSTAGE * 16;
};

// One 16-deep K block on the tensor pipe.  LA / LB are the shared-memory layouts of the tiles.
template <int MT, int LA, int LB, bool SCALE>
__device__ __forceinline__ void mma_block(double (&acc)[MT][MT][2], const double *as, const double *bs, int wm,
                                          int wn, int lane, int mi_valid, int nj_valid, double alpha) {
  using G = GemmCfg<MT>;
  const int r = lane >> 2, c = lane & 3;
  const double *pa = LA == 0 ? as + (wm * 8 * MT + r) * G::LD0 + c : as + c * G::LD1 + wm * 8 * MT + r;
  const double *pb = LB == 0 ? bs + (wn * 8 * MT + r) * G::LD0 + c : bs + c * G::LD1 + wn * 8 * MT + r;
#pragma unroll
  for (int ks = 0; ks < G::BK / 4; ++ks) {
    double af[MT], bf[MT];
#pragma unroll
    for (int i = 0; i < MT; ++i) {
      af[i] = LA == 0 ? pa[i * 8 * G::LD0 + ks * 4] : pa[ks * 4 * G::LD1 + i * 8];
      if (SCALE) af[i] *= alpha;
    }
#pragma unroll
    for (int j = 0; j < MT; ++j) bf[j] = LB == 0 ? pb[j * 8 * G::LD0 + ks * 4] : pb[ks * 4 * G::LD1 + j * 8];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
      for (int j = 0; j < MT; ++j)
        if (i < mi_valid && j < nj_valid) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
  }
}

// ROLE only names the instantiation (profiles list the launches by role): 0 integral contraction (a3),
// 1 rotation stage 1, 2 rotation stage 2 (a9), 3 H_eff stage 1 (a5), 4 H_eff stage 2 (a6).
template <int MT, int ROLE>
__global__ void __launch_bounds__(128) k_gemm_f64(const JobDesc *__restrict__ jobs,
                                                  const SegDesc *__restrict__ segs,
                                                  const TileDesc *__restrict__ tiles,
                                                  const __grid_constant__ BufTable bufs) {
  using G = GemmCfg<MT>;
  constexpr int BM = G::BM, BN = G::BN, BK = G::BK, EA = G::EA, EB = G::EB, NS = G::NSTAGE;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double *As = reinterpret_cast<double *>(smem_raw);
  double *Bs = As + NS * G::TILE_ELEMS;
  double *meta = Bs + NS * G::TILE_ELEMS;        // per stage: alpha, layout flags (as a double)

  const TileDesc td = tiles[blockIdx.x];
  const JobDesc jd = jobs[td.job];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, wm = warp & 1, wn = warp >> 1;
  const int m0 = td.m0, n0 = td.n0;
  const int Mrem = jd.M - m0, Nrem = jd.N - n0;   // > 0
  const int n1 = jd.n1;

  double acc[MT][MT][2];
#pragma unroll
  for (int i = 0; i < MT; ++i)
#pragma unroll
    for (int j = 0; j < MT; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
  int mi_valid = (Mrem - wm * 8 * MT + 7) / 8; mi_valid = max(0, min(MT, mi_valid));
  int nj_valid = (Nrem - wn * 8 * MT + 7) / 8; nj_valid = max(0, min(MT, nj_valid));

  // ---- producer state: set up once per segment, advanced by additions per K block
  int pseg = jd.seg_begin, pk0 = 0, pK = 0;
  const int seg_end = jd.seg_end;
  const double *pA = nullptr, *pB = nullptr;      // base of the current K block
  int64_t aoff[EA], boff[EB];                     // per-element offsets from pA / pB
  uint32_t adst[EA], bdst[EB];                    // per-element shared-memory byte offsets in a stage
  int ak[EA], bk[EB];                             // per-element k index inside the K block (-1: row/col out of range)
  int a_kq = 0, a_kr = 0, a_q16 = 0, a_r16 = 0, a_kn1 = FLAT_IDX, a_klo = 0, b_ks = 0, p_la = 0, p_lb = 0;
  int64_t a_khi = 0;
  double p_alpha = 1.0;
  const double *a_base = nullptr;
  const uint32_t smem_a = (uint32_t)__cvta_generic_to_shared(As), smem_b = (uint32_t)__cvta_generic_to_shared(Bs);

  auto setup_segment = [&]() {
    const SegDesc sd = segs[pseg];
    pK = sd.K; pk0 = 0; p_alpha = sd.alpha;
    a_base = rd_ref(bufs, sd.a);
    const double *Bp = rd_ref(bufs, sd.b);
    p_la = (sd.a_ms == 1 && sd.a_klo != 1) ? 1 : 0;
    p_lb = (sd.b_nlo == 1 && sd.b_ks != 1) ? 1 : 0;
    a_kn1 = sd.a_kn1; a_klo = sd.a_klo; a_khi = sd.a_khi; b_ks = sd.b_ks;
    if (p_la == 0) {                   // threads run along k: element j is (row tid/16 + 8j, k tid%16)
      const int kk = tid & 15;
      a_kq = kk / a_kn1; a_kr = kk - a_kq * a_kn1;
      a_q16 = BK / a_kn1; a_r16 = BK - a_q16 * a_kn1;
#pragma unroll
      for (int j = 0; j < EA; ++j) {
        const int mm = (tid >> 4) + 8 * j;
        aoff[j] = (int64_t)(m0 + mm) * sd.a_ms;
        adst[j] = (uint32_t)(mm * G::LD0 + kk) * 8u;
        ak[j] = mm < Mrem ? kk : -1;
      }
    } else {                           // threads run along m: element idx = tid + 128 j -> (m idx % BM, k idx / BM)
#pragma unroll
      for (int j = 0; j < EA; ++j) {
        const int idx = tid + 128 * j, mm = idx % BM, kk = idx / BM;
        const int kq = kk / a_kn1, kr = kk - kq * a_kn1;   // exact when the K block starts at a multiple of kn1 or k is flat
        aoff[j] = (int64_t)(m0 + mm) * sd.a_ms + (int64_t)kq * a_khi + (int64_t)kr * a_klo;
        adst[j] = (uint32_t)(kk * G::LD1 + mm) * 8u;
        ak[j] = mm < Mrem ? kk : -1;
      }
    }
    if (p_lb == 0) {                   // threads run along k
      const int kk = tid & 15;
#pragma unroll
      for (int j = 0; j < EB; ++j) {
        const int nn = (tid >> 4) + 8 * j, n = n0 + nn, nq = n / n1, nr = n - nq * n1;
        boff[j] = (int64_t)kk * sd.b_ks + (int64_t)nq * sd.b_nhi + (int64_t)nr * sd.b_nlo;
        bdst[j] = (uint32_t)(nn * G::LD0 + kk) * 8u;
        bk[j] = nn < Nrem ? kk : -1;
      }
    } else {                           // threads run along n
#pragma unroll
      for (int j = 0; j < EB; ++j) {
        const int idx = tid + 128 * j, nn = idx % BN, kk = idx / BN, n = n0 + nn, nq = n / n1, nr = n - nq * n1;
        boff[j] = (int64_t)kk * sd.b_ks + (int64_t)nq * sd.b_nhi + (int64_t)nr * sd.b_nlo;
        bdst[j] = (uint32_t)(kk * G::LD1 + nn) * 8u;
        bk[j] = nn < Nrem ? kk : -1;
      }
    }
    pA = a_base;
    pB = Bp;
  };

  // Issue the cp.async copies of the next K block into ring slot `stage` (always commits a group).
  auto produce = [&](int stage) {
    if (pseg < seg_end) {
      if (pk0 == 0 && pK == 0) setup_segment();
      const uint32_t sa = smem_a + stage * (G::TILE_ELEMS * 8), sb = smem_b + stage * (G::TILE_ELEMS * 8);
      const int krem = pK - pk0;
      const double *pa = p_la == 0 ? a_base + (int64_t)a_kq * a_khi + (int64_t)a_kr * a_klo : pA;
#pragma unroll
      for (int j = 0; j < EA; ++j) {
        const bool ok = ak[j] >= 0 && ak[j] < krem;
        cp_async8(sa + adst[j], ok ? pa + aoff[j] : a_base, ok);
      }
#pragma unroll
      for (int j = 0; j < EB; ++j) {
        const bool ok = bk[j] >= 0 && bk[j] < krem;
        cp_async8(sb + bdst[j], ok ? pB + boff[j] : a_base, ok);
      }
      if (tid == 0) { meta[stage * 2] = p_alpha; meta[stage * 2 + 1] = (double)(p_la * 2 + p_lb); }
      // advance to the next K block / segment
      pk0 += BK;
      if (pk0 >= pK) { ++pseg; pk0 = 0; pK = 0; }
      else {
        pB += (int64_t)BK * b_ks;
        if (p_la == 0) { a_kq += a_q16; a_kr += a_r16; if (a_kr >= a_kn1) { a_kr -= a_kn1; ++a_kq; } }
        else pA += (int64_t)BK * a_klo;    // layout 1 is only planned with a flat k index
      }
    }
    cp_async_commit();
  };

  const int n_iters = jd.n_iters;         // sum over segments of ceil(K / 16), from the plan
#pragma unroll
  for (int s = 0; s < NS - 1; ++s) produce(s);
  for (int it = 0; it < n_iters; ++it) {
    cp_async_wait<NS - 2>();
    __syncthreads();
    produce((it + NS - 1) % NS);
    const int stage = it % NS;
    const double *as = As + stage * G::TILE_ELEMS, *bs = Bs + stage * G::TILE_ELEMS;
    const double alpha = meta[stage * 2];
    const int lay = (int)meta[stage * 2 + 1];
    if (alpha == 1.0) {
      switch (lay) {
        case 0: mma_block<MT, 0, 0, false>(acc, as, bs, wm, wn, lane, mi_valid, nj_valid, alpha); break;
        case 1: mma_block<MT, 0, 1, false>(acc, as, bs, wm, wn, lane, mi_valid, nj_valid, alpha); break;
        case 2: mma_block<MT, 1, 0, false>(acc, as, bs, wm, wn, lane, mi_valid, nj_valid, alpha); break;
        default: mma_block<MT, 1, 1, false>(acc, as, bs, wm, wn, lane, mi_valid, nj_valid, alpha); break;
      }
    } else {
      switch (lay) {
        case 0: mma_block<MT, 0, 0, true>(acc, as, bs, wm, wn, lane, mi_valid, nj_valid, alpha); break;
        case 1: mma_block<MT, 0, 1, true>(acc, as, bs, wm, wn, lane, mi_valid, nj_valid, alpha); break;
        case 2: mma_block<MT, 1, 0, true>(acc, as, bs, wm, wn, lane, mi_valid, nj_valid, alpha); break;
        default: mma_block<MT, 1, 1, true>(acc, as, bs, wm, wn, lane, mi_valid, nj_valid, alpha); break;
      }
    }
  }
  cp_async_wait<0>();

  // epilogue: one write per element, optional per-column-group scale
  double *C = const_cast<double *>(rd_ref(bufs, jd.c));
  const double *scale = jd.scale >= 0 ? rd_ref(bufs, jd.scale) : nullptr;
#pragma unroll
  for (int j = 0; j < MT; ++j) {
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int nn = wn * 8 * MT + j * 8 + 2 * (lane & 3) + e;
      if (nn >= Nrem) continue;
      const int n = n0 + nn, nq = n / n1, nr = n - nq * n1;
      const double sc = scale ? __ldg(scale + nq) : 1.0;
      double *cp = C + (int64_t)nq * jd.c_nhi + (int64_t)nr * jd.c_nlo;
#pragma unroll
      for (int i = 0; i < MT; ++i) {
        const int mm = wm * 8 * MT + i * 8 + (lane >> 2);
        if (mm < Mrem) cp[(int64_t)(m0 + mm) * jd.c_ms] = acc[i][j][e] * sc;
      }
    }
  }
}

}  // namespace dmrg
