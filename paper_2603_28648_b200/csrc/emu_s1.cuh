// Stage 1 of the emulated-FP64 H_eff.psi (rows a4 + a5 of SURVEY.md 8(a)), second generation:
//   T[alpha][l][r'] = c_alpha sum_r psi[l][r] O_R,alpha[r'][r]      as  (operator lines (alpha, r')) x (psi rows l),
// written straight into the INT8 slices that stage 2 reads (and as FP64 only where an FP64 consumer exists).
//
// Why a kernel of its own (profiles/r1c_emu.md): K = d_R is only 2-6 k steps, so the generic
// segmented kernel spent ~2000 clk of MMAs and then ~14000 clk draining 384 TMEM columns per 128 x 64 tile, strictly
// one after the other.  Here
//   * a work item is one 128-line tile of a sliced right-operator unit; its A operand (all k steps, kappa slices,
//     <= 144 KB) is fetched ONCE into shared memory and stays resident while the item walks the psi rows of EVERY
//     job that uses the unit (all psi blocks with that right sector, all groups sharing the operators): the operator
//     slices are read from HBM once per unit instead of once per (job, tile);
//   * output tiles are 128 x 32, so two accumulator sets (kappa x 32 columns each) fit TMEM: the MMAs of tile t + 1
//     run while the epilogue drains tile t;
//   * the B slices of a k chunk are stacked along N (as in k_emu_seg), so the kappa (kappa + 1) / 2 slice products of
//     a k step are kappa MMAs 128 x (32 (kappa - s)) x 32;
//   * the epilogue takes the raw INT32 sums of its 16 columns into registers with six tcgen05.ld.x16, frees the set,
//     and produces the balanced digits of T without FP64 conversions: exact int64 joins -> 3 FMAs (radix-2^24
//     super-digits, reading s12) -> one multiply by the folded scale c_alpha 2^(eA + eB - e_T - BASE) ->
//     round-to-integer by the 1.5 * 2^52 add -> digit bytes by one 64-bit subtract and xor (emu_digit_bytes with the
//     bias folded into the subtrahend).
// Warp roles: warp 0 lane 0 issues the MMAs, warp 1 lane 0 issues the bulk copies, warps 2-9 are the epilogue
// (TMEM lane quarter = warp % 4, column half = (warp - 2) / 4).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <type_traits>

#include "emu_seg.cuh"

namespace dmrg {

constexpr int S1_BN = 32;                                     // psi rows per output tile
#ifndef S1_EPI_WARPS
#define S1_EPI_WARPS 8
#endif
constexpr int S1_EPI = S1_EPI_WARPS;                          // epilogue warps: 8 (16 columns each) or 16 (8 columns each)
constexpr int S1_CPW = S1_BN / (S1_EPI / 4);                 // columns per epilogue warp
constexpr int S1_THREADS = 64 + 32 * S1_EPI;
__host__ __device__ constexpr int s1_kres(int kappa) { return kappa <= 6 ? 6 : 5; }     // resident k steps of A
__host__ __device__ constexpr int s1_smem_bytes(int kappa) {
  return s1_kres(kappa) * kappa * (EMU_BM * 32) + 2 * s1_kres(kappa) * kappa * (S1_BN * 32);
}

__device__ __forceinline__ void tmem_ld16_nowait(uint32_t taddr, int32_t (&v)[16]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                 "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
               : "r"(taddr) : "memory");
}

__device__ __forceinline__ void tmem_ld4_nowait(uint32_t taddr, int32_t (&v)[4]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];\n"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(taddr) : "memory");
}

// a * b + c with a 64-bit result in ONE instruction (SASS IMAD.WIDE): the exact joins of the INT32 sums
__device__ __forceinline__ long long mad_wide(int a, int b, long long c) {
  long long d;
  asm("mad.wide.s32 %0, %1, %2, %3;\n" : "=l"(d) : "r"(a), "r"(b), "l"(c));
  return d;
}
// MAGIC + p[lo] + 2^8 p[lo-1] + 2^16 p[lo-2]: a radix-2^24 super-digit (|G| < 2^48) already carrying the bits of
// 1.5 * 2^52, so that reinterpreting it as a double gives 1.5 * 2^52 + G exactly
// (the multipliers m0 = 1, m8 = 2^8, m16 = 2^16 come in registers that ptxas cannot see through: with literal
// constants it strength-reduces each mad.wide into five shift / add-with-carry instructions)
template <int KAPPA, int NC>
__device__ __forceinline__ double s1_join3(const int32_t (&pv)[KAPPA][NC], int lo, int e, int m0, int m8, int m16) {
  long long G = mad_wide(pv[lo][e], m0, 0x4338000000000000LL);
  if (lo >= 1) G = mad_wide(pv[lo - 1][e], m8, G);
  if (lo >= 2) G = mad_wide(pv[lo - 2][e], m16, G);
  return __longlong_as_double(G);
}
// Byte transpose of the digit bytes of 4 consecutive k: xl / xh = low / high word of each element's digit bytes
// (digit i = byte i), w[slice] = the 4 digits of slice kappa - 1 - i.  12 PRMT at kappa = 6 (emu_pack4: 18).
template <int KAPPA>
__device__ __forceinline__ void s1_pack4(const uint32_t (&xl)[4], const uint32_t (&xh)[4], uint32_t (&w)[KAPPA]) {
  const uint32_t a_lo = __byte_perm(xl[0], xl[1], 0x5140), b_lo = __byte_perm(xl[2], xl[3], 0x5140);
  w[KAPPA - 1] = __byte_perm(a_lo, b_lo, 0x5410);
  w[KAPPA - 2] = __byte_perm(a_lo, b_lo, 0x7632);
  if constexpr (KAPPA >= 3) {
    const uint32_t a_hi = __byte_perm(xl[0], xl[1], 0x7362), b_hi = __byte_perm(xl[2], xl[3], 0x7362);
    w[KAPPA - 3] = __byte_perm(a_hi, b_hi, 0x5410);
    if constexpr (KAPPA >= 4) w[KAPPA - 4] = __byte_perm(a_hi, b_hi, 0x7632);
  }
  if constexpr (KAPPA >= 5) {
    const uint32_t c_lo = __byte_perm(xh[0], xh[1], 0x5140), d_lo = __byte_perm(xh[2], xh[3], 0x5140);
    w[KAPPA - 5] = __byte_perm(c_lo, d_lo, 0x5410);
    if constexpr (KAPPA >= 6) w[KAPPA - 6] = __byte_perm(c_lo, d_lo, 0x7632);
    if constexpr (KAPPA >= 7) {
      const uint32_t c_hi = __byte_perm(xh[0], xh[1], 0x7362), d_hi = __byte_perm(xh[2], xh[3], 0x7362);
      w[KAPPA - 7] = __byte_perm(c_hi, d_hi, 0x5410);
    }
  }
}

template <int KAPPA>
__global__ void __launch_bounds__(S1_THREADS, 1) k_emu_s1(const EmuS1Item *__restrict__ items, const int *__restrict__ cta_begin,
                                                          const EmuS1Tile *__restrict__ ntiles, const EmuJob *__restrict__ jobs,
                                                          BufTable bufs, const int8_t *__restrict__ slA,
                                                          const int8_t *__restrict__ slB, const int32_t *__restrict__ exA,
                                                          const int32_t *__restrict__ exB, int8_t *__restrict__ fuse_sl,
                                                          int32_t *__restrict__ fuse_ex, const double *__restrict__ norms) {
  constexpr int KRES = s1_kres(KAPPA);
  constexpr int A_SLICE = EMU_BM * 32, A_STEP = KAPPA * A_SLICE;         // bytes of one slice / one k step of the A tile
  constexpr int B_SLICE = S1_BN * 16, B_STEP = KAPPA * S1_BN * 32;       // one slice of one k chunk / one k step of a B tile
  constexpr int B_BUF = KRES * B_STEP;
  constexpr int T_SLICE = 2 * EMU_BN * 16;                               // stage-2 operand: 64-row tiles (emu_seg.cuh)
  constexpr int BASE = 8 * KAPPA - 2;
  constexpr int SET_COLS = KAPPA * S1_BN;
  extern __shared__ __align__(128) unsigned char smem[];
  __shared__ __align__(8) uint64_t bar_afull, bar_aempty, bar_bfull[2], bar_bempty[2], bar_done[2], bar_tfree[2];
  __shared__ uint32_t tmem_slot;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t smem_a = (uint32_t)__cvta_generic_to_shared(smem), smem_b = smem_a + KRES * A_STEP;

  if (warp == 0) tmem_alloc(&tmem_slot, 512);
  if (tid == 0) {
    mbar_init(&bar_afull, 1); mbar_init(&bar_aempty, 1);
    for (int s = 0; s < 2; ++s) {
      mbar_init(&bar_bfull[s], 1); mbar_init(&bar_bempty[s], 1); mbar_init(&bar_done[s], 1); mbar_init(&bar_tfree[s], S1_EPI);
    }
  }
  asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
  const uint32_t tmem = tmem_slot;
  const int i_begin = cta_begin[blockIdx.x], i_end = cta_begin[blockIdx.x + 1];

  if (warp == 0) {
    // ---------------------------------------------------------------- MMA issuer (all lanes walk the lists, one issues:
    // tc_i8.cuh elect_one)
    {
      const bool leader = elect_one();
      uint32_t ph_afull = 0, ph_bfull = 0, ph_tfree = 0;
      int cnt = 0;                                       // tiles issued so far: set = buffer = cnt & 1
      for (int i = i_begin; i < i_end; ++i) {
        const EmuS1Item it = items[i];
        mbar_wait(&bar_afull, ph_afull); ph_afull ^= 1u;
        for (int t = it.nt_begin; t < it.nt_end; ++t, ++cnt) {
          const int set = cnt & 1;
          if (cnt >= 2) { mbar_wait(&bar_tfree[set], (ph_tfree >> set) & 1u); ph_tfree ^= 1u << set; }
          mbar_wait(&bar_bfull[set], (ph_bfull >> set) & 1u); ph_bfull ^= 1u << set;
          asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
          for (int k = 0; k < it.ksteps; ++k) {
            const uint32_t sa = smem_a + k * A_STEP, sb = smem_b + set * B_BUF + k * B_STEP;
            const uint64_t da = umma_smem_desc(sa, EMU_BM * 16, 128), db = umma_smem_desc(sb, KAPPA * B_SLICE, 128);
            if (leader) {
#pragma unroll
              for (int s = 0; s < KAPPA; ++s)          // A slice s x B slices 0 .. kappa-1-s -> accumulators s .. kappa-1
                umma_i8(tmem + (uint32_t)(set * SET_COLS + s * S1_BN), da + (uint64_t)((s * A_SLICE) >> 4), db,
                        umma_idesc_s8(EMU_BM, S1_BN * (KAPPA - s)), !(k == 0 && s == 0));
            }
            __syncwarp();
          }
          if (leader) {
            umma_commit(&bar_bempty[set]);
            umma_commit(&bar_done[set]);
          }
          __syncwarp();
        }
        if (leader) umma_commit(&bar_aempty);            // every MMA that reads this A tile has completed
        __syncwarp();
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // ---------------------------------------------------------------- producer
    if (lane == 0) {
      uint32_t ph_aempty = 0, ph_bempty = 0;
      int cnt = 0;
      for (int i = i_begin; i < i_end; ++i) {
        const EmuS1Item it = items[i];
        if (i > i_begin) { mbar_wait(&bar_aempty, ph_aempty); ph_aempty ^= 1u; }
        mbar_expect_tx(&bar_afull, (uint32_t)(it.ksteps * A_STEP));
        const int8_t *ga = slA + it.a_off * KAPPA;
        for (int k = 0; k < it.ksteps; ++k) bulk_g2s(smem_a + k * A_STEP, ga + (int64_t)k * A_STEP, A_STEP, &bar_afull);
        for (int t = it.nt_begin; t < it.nt_end; ++t, ++cnt) {
          const int set = cnt & 1;
          if (cnt >= 2) { mbar_wait(&bar_bempty[set], (ph_bempty >> set) & 1u); ph_bempty ^= 1u << set; }
          const uint32_t bytes = (uint32_t)(it.ksteps * B_STEP);
          mbar_expect_tx(&bar_bfull[set], bytes);
          bulk_g2s(smem_b + set * B_BUF, slB + ntiles[t].b_off * KAPPA, bytes, &bar_bfull[set]);
        }
      }
    }
    __syncwarp();
  } else {
    // ---------------------------------------------------------------- epilogue
    // Per tile and thread: 16 columns (psi rows l) of one line (alpha, r'), taken from TMEM in batches of 4 so that
    // only 48 raw sums are live (two batches: one being recombined, one in flight).  Everything that depends on the JOB (coefficient, exponent of the T line, target
    // addresses) is set up once per job: consecutive n-tiles of an item belong to the same job ~3-4 times in a row.
    constexpr int CPW = S1_CPW;
    const int quarter = warp & 3, half = (warp - 2) >> 2, trow = quarter * 32 + lane;      // half: column group of CPW
    const uint32_t tbase = tmem + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(half * CPW);
    constexpr uint64_t DIGIT_BIAS = 0x8080808080808080ull >> (8 * (9 - KAPPA));
    constexpr long long MAGIC = 0x4338000000000000LL;             // bits of 1.5 * 2^52
    // 1.5 * 2^52 + digit bias: the add rounds Y to an integer and leaves (Y + BIAS) in the low mantissa bits, whose
    // bytes are the balanced digits + 128 (emu_digit_bytes); the xor that removes the 128 is applied after packing
    const double C1 = __longlong_as_double(MAGIC + (long long)DIGIT_BIAS);
    double wc[KAPPA];
#pragma unroll
    for (int c = 0; c < KAPPA; ++c) wc[c] = scalbn(1.0, 16 * KAPPA - 8 * (c + 2));
    const double wneg = -6755399441055744.0 * wc[KAPPA - 1];
    int m0, m8, m16;                                      // 1, 2^8, 2^16 in registers (see s1_join3)
    asm volatile("mov.u32 %0, 1;\n mov.u32 %1, 256;\n mov.u32 %2, 65536;\n" : "=r"(m0), "=r"(m8), "=r"(m16));
    uint32_t ph_done = 0;
    int cnt = 0;
    for (int i = i_begin; i < i_end; ++i) {
      const EmuS1Item it = items[i];
      const int row = it.m0 + trow;
      const bool row_ok = row < it.lines;
      const int eA = row_ok ? exA[it.ea_off + row] : 0;
      const int r_hi = row / it.n1, r_lo = row - r_hi * it.n1;      // member alpha and line r' (n1 = d_R' of the unit)
      // job state
      int cur_job = -1, N = 0, lim = 0, fuse = 0, want64 = 0, rs_hib = 0, rs_lo = 0, koff = 0, padk = -1;
      int64_t ldc = 0;
      double f64 = 1.0;
      int8_t *unit = nullptr;
      double *Crow = nullptr;
      EmuS1Tile tl = ntiles[it.nt_begin];
      for (int t = it.nt_begin; t < it.nt_end; ++t, ++cnt) {
        const int set = cnt & 1;
        const EmuS1Tile cur = tl;
        if (t + 1 < it.nt_end) tl = ntiles[t + 1];              // prefetch the next descriptor
        if (cur.job != cur_job) {
          cur_job = cur.job;
          const EmuJob *jb = jobs + cur.job;
          N = jb->N; fuse = jb->fuse;
          const int dlpad = jb->dlpad;
          lim = fuse ? dlpad : N;
          want64 = !fuse || jb->write_fp64;
          // folded scale of this thread's line: c_alpha 2^(eA - e_T) takes the integer value of the product to the
          // digits of T (exponent e_T = the bound of reading s12b, known before the product); 2^(e_T - BASE) to FP64
          double coef = 1.0;
          const ref_t sref = jb->scale;
          if (sref >= 0 && row_ok) coef = (bufs.p[sref >> 48] + (sref & REF_MASK))[r_hi];
          int e_T = 0;
          if (fuse && row_ok) {
            const double bnd = norms[jb->psi_blk] * norms[jb->qn_off + r_lo] * (1.0 + 0x1p-20);
            if (bnd > 0.0) frexp(bnd, &e_T);
          }
          const double rs = coef * pow2i(fuse ? eA - e_T : eA - BASE);                 // !fuse: straight to FP64
          f64 = fuse ? pow2i(e_T - BASE) : 1.0;
          // the column scale rs 2^(eB_l - BASE) is formed by an add on the exponent field (the exponents met here are
          // far inside the normal range); rs = 0 keeps a zero high word: a denormal scale whose digits round to 0
          rs_hib = rs != 0.0 ? __double2hiint(rs) - (BASE << 20) : 0;
          rs_lo = __double2loint(rs);
          ldc = jb->c_ld;
          Crow = bufs.p[jb->c >> 48] + (jb->c & REF_MASK) + r_lo + (int64_t)r_hi * jb->c_nhi;
          if (fuse) {
            // slices of T for stage 2: line r' of the unit of member alpha, K index = member * dlpad + l (layout of
            // emu_seg.cuh, 64-row tiles): this thread writes one aligned 16-byte chunk per slice and tile
            const int per_piece = jb->per_piece, n_pieces = jb->n_pieces;
            const int pc = r_hi < per_piece ? 0 : r_hi / per_piece, a_loc = r_hi - pc * per_piece;
            const int ksteps_pc = (pc == n_pieces - 1 ? jb->ld_last : jb->ld_full) >> 5;
            unit = fuse_sl + (jb->t_out_off + (int64_t)pc * jb->piece_bytes + (int64_t)(r_lo >> 6) * ksteps_pc * T_SLICE) * KAPPA +
                   (r_lo & 63) * 16;
            koff = a_loc * dlpad;
            if (half == 0 && row_ok) fuse_ex[jb->t_exp_off + (int64_t)pc * it.n1 + r_lo] = e_T;
            // the chunk that pads the unit's K to a multiple of 32 is zeroed by the thread that writes the last chunk
            const int members = it.lines / it.n1;
            const int na = pc == n_pieces - 1 ? members - pc * per_piece : per_piece;
            padk = (a_loc == na - 1 && ((na * dlpad) & 31) == 16) ? na * dlpad : -1;
          }
        }
        const int l0 = cur.n0 + half * CPW;
        // exponents of the 16 psi rows (segments are 16-byte aligned, plan_heff_jobs.cpp); columns past N carry
        // whatever follows: their digits meet zero digits of the left operators in stage 2
        int ecol[CPW];
        {
          const int4 *ep = reinterpret_cast<const int4 *>(exB + cur.eb_off + l0);
#pragma unroll
          for (int g = 0; g < CPW / 4; ++g) { const int4 q = ep[g]; ecol[4 * g] = q.x; ecol[4 * g + 1] = q.y; ecol[4 * g + 2] = q.z; ecol[4 * g + 3] = q.w; }
        }
        mbar_wait(&bar_done[set], (ph_done >> set) & 1u); ph_done ^= 1u << set;
        __syncwarp();                                           // lanes that skipped the last tile's stores rejoin here
        asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory");
        const bool active = row_ok && l0 < lim;
        // The raw sums come out of TMEM four columns at a time into two register buffers: the loads of batch b + 1 are in
        // flight while batch b is recombined (the epilogue warps are latency bound: 2 per scheduler)
        uint32_t w[CPW / 4][KAPPA];
        // the FP64 copy of T is wanted by few jobs: its stores, products and address arithmetic are compiled into a second
        // version of the drain instead of being predicated off 16 times per tile in the common one
        auto drain = [&](auto W64) {
        constexpr bool w64 = decltype(W64)::value;
        int32_t pv[2][KAPPA][4];
#pragma unroll
        for (int c = 0; c < KAPPA; ++c) tmem_ld4_nowait(tbase + (uint32_t)(set * SET_COLS + c * S1_BN), pv[0][c]);
#pragma unroll
        for (int b = 0; b < CPW / 4; ++b) {
          tmem_ld_wait();                                       // batch b has landed
          if (b + 1 < CPW / 4) {
#pragma unroll
            for (int c = 0; c < KAPPA; ++c)
              tmem_ld4_nowait(tbase + (uint32_t)(set * SET_COLS + c * S1_BN + (b + 1) * 4), pv[(b + 1) & 1][c]);
          } else {                                              // every raw sum is in registers: the set may be overwritten
            asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_tfree[set]);
          }
          if (active) {
            uint32_t xl[4], xh[4];
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {
              const int e = 4 * b + jj;
              // exact joins of three neighbouring anti-diagonal sums into radix-2^24 super-digits (|G| < 2^48), exact
              // conversion by the magic number, super-digits summed in FP64 smallest scale first (reading s12)
              double v = fma(s1_join3<KAPPA, 4>(pv[b & 1], KAPPA - 1, jj, m0, m8, m16), wc[KAPPA - 1], wneg);
#pragma unroll
              for (int lo = KAPPA - 4; lo >= 0; lo -= 3)
                v = fma(s1_join3<KAPPA, 4>(pv[b & 1], lo, jj, m0, m8, m16) - 6755399441055744.0, wc[lo], v);
              const double y = v * __hiloint2double(rs_hib == 0 ? 0 : rs_hib + (ecol[e] << 20), rs_lo);
              if constexpr (w64) {
                if (l0 + e < N) Crow[(int64_t)(l0 + e) * ldc] = y * f64;             // consecutive lanes = consecutive addresses
              }
              if constexpr (KAPPA <= 6) {          // |Y| < 2^46: the magic add is exact
                const long long zb = __double_as_longlong(y + C1);
                xl[jj] = (uint32_t)zb; xh[jj] = (uint32_t)(zb >> 32);
              } else {                             // kappa = 7: |Y| < 2^54 does not fit the mantissa trick
                const uint64_t ub = emu_digit_bytes<KAPPA>(llrint(y));
                xl[jj] = (uint32_t)ub; xh[jj] = (uint32_t)(ub >> 32);
              }
            }
            s1_pack4<KAPPA>(xl, xh, w[b]);
            if constexpr (KAPPA <= 6) {
#pragma unroll
              for (int sl = 1; sl < KAPPA; ++sl) w[b][sl] ^= 0x80808080u;   // all digits but the top one carry + 128
            }
          }
        }
        };
        if (want64) drain(std::true_type()); else drain(std::false_type());
        if (!active || !fuse) continue;
        const int k = koff + l0;
        int8_t *dst = unit + (int64_t)(k >> 5) * (T_SLICE * KAPPA) + ((k >> 4) & 1) * (KAPPA * EMU_BN * 16);
#pragma unroll
        for (int sl = 0; sl < KAPPA; ++sl) {
          if constexpr (CPW == 16) *reinterpret_cast<uint4 *>(dst + sl * (EMU_BN * 16)) = make_uint4(w[0][sl], w[1][sl], w[2][sl], w[3][sl]);
          else *reinterpret_cast<uint2 *>(dst + sl * (EMU_BN * 16) + (k & 8)) = make_uint2(w[0][sl], w[1][sl]);   // half a chunk
        }
        if (k + CPW == padk) {
          int8_t *d2 = unit + (int64_t)(padk >> 5) * (T_SLICE * KAPPA) + ((padk >> 4) & 1) * (KAPPA * EMU_BN * 16);
#pragma unroll
          for (int sl = 0; sl < KAPPA; ++sl) *reinterpret_cast<uint4 *>(d2 + sl * (EMU_BN * 16)) = make_uint4(0u, 0u, 0u, 0u);
        }
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory");
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 512);
}

}  // namespace dmrg
