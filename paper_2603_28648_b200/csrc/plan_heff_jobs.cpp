// Stage-1 / stage-2 / diagonal descriptors of the H_eff plan.
//   stage 1:  T[alpha][l][r'] = c_alpha sum_r psi[l][r] O_R,alpha[r'][r]      (one job per run, psi block, r' sector)
//   stage 2:  psi'[b'][l'][r'] += G sum_{alpha,l} O_L,alpha[l'][l] T[alpha][l][r']
// G is the geometry factor of (group, b -> b'): the fermion sign of Appendix A5 for U(1)xU(1); for
// SU(2) the product F6 F9_A F9_B of 9j prefactors with the signs (-1)^{N_1 pi_U} and the tilde
// factors of daggered block operators.  It multiplies the stage-2 segment, so T is shared by all b'.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <map>
#include <stdexcept>
#include <tuple>

#include "internal.h"

namespace dmrg {

namespace {
inline bool tri2(int a, int b, int c) { return c >= std::abs(a - b) && c <= a + b && ((a + b + c) % 2) == 0; }
inline bool nine_j_allowed(int j1, int j2, int J, int k1, int k2, int K, int j1p, int j2p, int Jp) {   // rows and columns
  return tri2(j1, j2, J) && tri2(k1, k2, K) && tri2(j1p, j2p, Jp) && tri2(j1, k1, j1p) && tri2(j2, k2, j2p) && tri2(J, K, Jp);
}
inline double tilde_factor(int S_bra, int S_ket, int k2) {   // <bra||T~||ket> = factor * <ket||T||bra>
  int e = (S_ket - S_bra + k2) / 2;
  return ((e & 1) ? -1.0 : 1.0) * std::sqrt((S_ket + 1.0) / (S_bra + 1.0));
}
// bra sectors reachable from ket sector q by an operator of class (dN, second)
std::vector<int> bra_sectors(const BondTable &t, int sym, const Sector &q, DQ dq) {
  std::vector<int> r;
  if (sym == 0) { int i = t.find(q.N + dq.dN, q.S + dq.dS); if (i >= 0) r.push_back(i); return r; }
  for (int S2 = std::abs(q.S - dq.dS); S2 <= q.S + dq.dS; S2 += 2) {
    int i = t.find(q.N + dq.dN, S2);
    if (i >= 0) r.push_back(i);
  }
  return r;
}
}  // namespace

void build_heff_jobs(HeffPlan &P, const BlockState &Lb, const BlockState &Rb, int N, int twoS, int BM, int BN) {
  const int sym = Lb.sym;
  std::vector<std::vector<SegDesc>> segs2(P.psi.size());
  std::vector<std::vector<int>> segn2(P.psi.size());   // members per stage-2 segment
  std::vector<std::vector<int>> segp2(P.psi.size());   // pass of each stage-2 segment
  // The intermediate T of a whole apply can exceed HBM (188 GB at configs[3]); the apply is cut into
  // passes whose T fits `scratch_budget`; every pass runs its stage-1 jobs, then its stage-2 chunks.
  const int64_t budget = std::max<int64_t>(P.scratch_budget, 1);
  int pass = 0;
  int64_t max_scratch = 0;
  P.stage1v.assign(1, JobList());
  std::vector<std::vector<DiagTerm>> diag(P.psi.size());
  int64_t scratch = 0;
  P.tab_falg_blocks.assign(P.psi.size(), 0);
  // Emulated mode: a two-sided stage-2 segment whose operands are large enough is cut at member boundaries
  // into pieces of K <= 16384 (INT32 accumulators of up to 7 products of 2^14 cannot overflow); every piece
  // is one EmuSeg with its own exponent sets.  Left operator pieces are sliced once per bond and shared by
  // all psi blocks that use them; T pieces are sliced after stage 1 of their pass.
  std::vector<std::vector<EmuSeg>> esegs2(P.psi.size());
  std::vector<std::vector<int>> epass2(P.psi.size());
  std::map<std::tuple<ref_t, int, int>, int> lunits;      // (address, dagger, members) -> first piece in sliceL
  P.emu.assign(1, EmuPass());
  std::map<std::tuple<ref_t, int, int, int64_t>, int64_t> qnorms;   // (address, dagger, members, coef) -> norms offset
  P.emu_norm_elems = (int64_t)P.psi.size();
  const bool emu_bound = P.opt.emu_exact_exp == 0;
  const bool emu_fuse = P.opt.emu_fuse != 0;     // stage-1 epilogue emits the slices of T
  // emulated stage 1: T^T = coef * O_R psi[b]^T with A = the stacked right operators, lines (member, r') (sliced
  // once per bond) and B = the psi block, lines l (sliced every apply)
  const bool emu_stage1 = P.emu_mode && P.opt.emu_stage1 != 0;
  const int emu_minM1 = P.opt.emu_minm1, emu_minK1 = P.opt.emu_mink1,
            emu_minN1 = P.opt.emu_minn1;
  std::vector<int> punit(P.psi.size(), -1);                        // psi block -> index in sliceP (64-row tiles, k_emu_seg)
  std::vector<int> punit32(P.psi.size(), -1);                      // psi block -> index in sliceP (32-row tiles, k_emu_s1)
  // second-generation stage-1 kernel (emu_s1.cuh): jobs whose K fits its resident A tile
  const bool emu_s1new = emu_stage1 && !P.emu_tf32 && P.opt.emu_s1new != 0;
  const int s1_kres = P.kappa <= 6 ? 6 : 5;
  std::map<std::tuple<ref_t, int, int>, std::pair<int64_t, int64_t>> runits;   // right unit -> (out_off, exp_off)
  int64_t emuT_cur = 0, expT_cur = 0;
  // emu_minm = 0 (default): 8 when the largest sector of the two blocks reaches 96, else 32.  A narrow output block wastes
  // most of a 128-row MMA, yet on systems with large sectors the tensor path still beats the FP64 remainder kernel 4 : 1
  // (configs[2]: 53.3 -> 50.9 ms per apply); on systems of small sectors (configs[4], median 10) the FP64 kernel on 32 x 32
  // tiles wins (1020 vs 1075 ms).
  int64_t maxdim = 1;
  for (const Sector &sc : Lb.tab.sec) maxdim = std::max(maxdim, sc.dim);
  for (const Sector &sc : Rb.tab.sec) maxdim = std::max(maxdim, sc.dim);
  const int emu_minK = P.opt.emu_mink, emu_minM = P.opt.emu_minm ? P.opt.emu_minm : (maxdim >= 96 ? 8 : 32),
            emu_minN = P.opt.emu_minn;
  for (const Group &g : P.groups) {
    const int kindL = Lb.classes[g.clsL].kind, kindR = Rb.classes[g.clsR].kind;
    const int kL = Lb.classes[g.clsL].dq.dS, kR = Rb.classes[g.clsR].dq.dS;     // SU(2): doubled ranks
    const int pi1 = (site_N(sym, g.s1p) - site_N(sym, g.s1)) & 1, pi2 = (site_N(sym, g.s2p) - site_N(sym, g.s2)) & 1;
    const int piR = g.dqR.dN & 1;
    for (size_t bi = 0; bi < P.psi.size(); ++bi) {
      const PsiBlock &b = P.psi[bi];
      if (b.s1 != g.s1 || b.s2 != g.s2) continue;
      const Sector &qL = Lb.tab.sec[b.iL], &qR = Rb.tab.sec[b.iR];
      const int64_t dL = b.dL, dR = b.dR;
      for (int iRp : bra_sectors(Rb.tab, sym, qR, g.dqR)) {
        const int64_t dRp = Rb.tab.sec[iRp].dim;
        const int rbra = g.dagR ? b.iR : iRp, rket = g.dagR ? iRp : b.iR;   // stored orientation
        // one stage-1 job per run for this (b, iRp), created lazily when some output uses it
        std::vector<int64_t> toff(g.runs.size(), -1);
        std::vector<int> tpass(g.runs.size(), 0);
        std::vector<int> tuni(g.runs.size(), -1);           // first piece of the T job in emu[pass].sliceT
        int64_t maxLp = 0;
        for (int iLp : bra_sectors(Lb.tab, sym, qL, g.dqL)) maxLp = std::max<int64_t>(maxLp, Lb.tab.sec[iLp].dim);
        const int dlpad = (int)((dL + 15) / 16 * 16);                  // stage-2 K index = member * dlpad + l
        const int per_piece = std::max(1, P.opt.emu_kpiece / dlpad);   // members per piece: K <= 16384 (option emu_kpiece)
        std::vector<int> ej1(g.runs.size(), -1);                       // emulated stage-1 job of the run (in emu[tpass].jobs1)
        for (int iLp : bra_sectors(Lb.tab, sym, qL, g.dqL)) {
          const int64_t dLp = Lb.tab.sec[iLp].dim;
          const int lbra = g.dagL ? b.iL : iLp, lket = g.dagL ? iLp : b.iL;
          const int SLp = Lb.tab.sec[iLp].S, SRp = Rb.tab.sec[iRp].S;
          for (int SAp : fuse_S(sym, SLp, g.s1p))
            for (int SBp : fuse_S(sym, SRp, g.s2p)) {
              auto po = P.psi_index.find(std::make_tuple(iLp, g.s1p, SAp, g.s2p, iRp, SBp));
              if (po == P.psi_index.end()) continue;
              double G;
              if (sym == 0) {   // Appendix A5 sign: (-1)^{N_l(pi1+pi2+piR) + N_s1(pi2+piR) + N_s2 piR}
                int e = qL.N * (pi1 + pi2 + piR) + site_N(sym, b.s1) * (pi2 + piR) + site_N(sym, b.s2) * piR;
                G = (e & 1) ? -1.0 : 1.0;
              } else {
                // a block pair is coupled when the triangle conditions of the three 9j symbols hold (the definition
                // F_alg counts by); an accidental zero of a symbol is executed with G = 0
                if (!nine_j_allowed(qL.S, site_S(sym, g.s1), b.SA, kL, g.k1, g.kk, SLp, site_S(sym, g.s1p), SAp) ||
                    !nine_j_allowed(site_S(sym, g.s2), qR.S, b.SB, g.k2, kR, g.kk, site_S(sym, g.s2p), SRp, SBp) ||
                    !nine_j_allowed(b.SA, b.SB, twoS, g.kk, g.kk, 0, SAp, SBp, twoS)) continue;
                double fa = su2_f9(qL.S, site_S(sym, g.s1), b.SA, kL, g.k1, g.kk, SLp, site_S(sym, g.s1p), SAp);
                double fb = su2_f9(site_S(sym, g.s2), qR.S, b.SB, g.k2, kR, g.kk, site_S(sym, g.s2p), SRp, SBp);
                double f6 = su2_f9(b.SA, b.SB, twoS, g.kk, g.kk, 0, SAp, SBp, twoS);
                G = fa * fb * f6;
                int e = qL.N * pi1 + site_N(sym, b.s2) * piR + (qL.N + site_N(sym, b.s1)) * ((pi2 + piR) & 1);
                if (e & 1) G = -G;
                if (g.dagL) G *= tilde_factor(SLp, qL.S, kL);
                if (g.dagR) G *= tilde_factor(SRp, qR.S, kR);
              }
              const int bo = po->second;
              const bool diagonal = (bo == (int)bi);
              for (size_t ri = 0; ri < g.runs.size(); ++ri) {
                const Run &r = g.runs[ri];
                ref_t la, ra;
                if (!op_addr(P.resL, r.L, B_OPS_L, B_DER_L, lbra, lket, &la, nullptr)) continue;
                if (!op_addr(P.resR, r.R, B_OPS_R, B_DER_R, rbra, rket, &ra, nullptr)) continue;
                if (diagonal)
                  for (int a = 0; a < r.n; ++a)
                    diag[bi].push_back({la + a * dL * dL, ra + a * dR * dR, (int32_t)(dL + 1), (int32_t)(dR + 1),
                                        G * r.c[a]});
                SegDesc sg{};
                if (kindR == K_I) {            // one-sided left: psi'[l'][r] += f O_L[l'][l] psi[l][r]
                  if (r.n != 1) throw std::logic_error("one-sided run with n > 1");
                  sg.a = la; sg.K = (int32_t)dL; sg.a_kn1 = FLAT; sg.a_khi = 0;
                  if (!g.dagL) { sg.a_ms = (int32_t)dL; sg.a_klo = 1; } else { sg.a_ms = 1; sg.a_klo = (int32_t)dLp; }
                  sg.b = mkref(B_PSI_IN, b.off); sg.b_ks = (int32_t)dR; sg.b_nlo = 1; sg.b_nhi = 0;
                  sg.alpha = G * r.c[0];
                  segs2[bo].push_back(sg); segn2[bo].push_back(1); segp2[bo].push_back(pass);
                  P.falg += 2 * dLp * dL * dR;
                  P.flops2 += 2 * dLp * dL * dR;
                  P.tab_falg_blocks[bo] += 2 * dLp * dL * dR;
                  continue;
                }
                if (kindL == K_I) {            // one-sided right: psi'[l][r'] += f psi[l][r] O_R[r'][r]
                  if (r.n != 1) throw std::logic_error("one-sided run with n > 1");
                  sg.a = mkref(B_PSI_IN, b.off); sg.a_ms = (int32_t)dR; sg.a_kn1 = FLAT; sg.a_klo = 1; sg.a_khi = 0;
                  sg.K = (int32_t)dR;
                  sg.b = ra; sg.b_nhi = 0;
                  if (!g.dagR) { sg.b_ks = 1; sg.b_nlo = (int32_t)dR; } else { sg.b_ks = (int32_t)dRp; sg.b_nlo = 1; }
                  sg.alpha = G * r.c[0];
                  segs2[bo].push_back(sg); segn2[bo].push_back(1); segp2[bo].push_back(pass);
                  P.falg += 2 * dL * dR * dRp;
                  P.flops2 += 2 * dL * dR * dRp;
                  P.tab_falg_blocks[bo] += 2 * dL * dR * dRp;
                  continue;
                }
                if (toff[ri] < 0) {            // stage 1 for (run, b, iRp), shared by every output block
                  const int64_t need = (int64_t)r.n * dL * dRp;
                  if (scratch > 0 && scratch + need > budget) {
                    ++pass; scratch = 0; P.stage1v.push_back(JobList());
                    P.emu.push_back(EmuPass()); emuT_cur = 0; expT_cur = 0;
                  }
                  toff[ri] = scratch; tpass[ri] = pass;
                  scratch += need;
                  max_scratch = std::max(max_scratch, scratch);
                  SegDesc s1{};
                  s1.a = mkref(B_PSI_IN, b.off); s1.a_ms = (int32_t)dR; s1.a_kn1 = FLAT; s1.a_klo = 1; s1.a_khi = 0;
                  s1.K = (int32_t)dR; s1.alpha = 1.0; s1.b = ra;
                  if (!g.dagR) { s1.b_ks = 1; s1.b_nlo = (int32_t)dR; s1.b_nhi = dRp * dR; }
                  else { s1.b_ks = (int32_t)dRp; s1.b_nlo = 1; s1.b_nhi = dR * dRp; }
                  JobDesc j1{};
                  j1.c = mkref(B_SCRATCH, toff[ri]); j1.scale = mkref(B_COEF, r.coef_off);
                  j1.M = (int32_t)dL; j1.N = (int32_t)(r.n * dRp); j1.c_ms = (int32_t)dRp; j1.n1 = (int32_t)dRp;
                  j1.c_nlo = 1; j1.c_nhi = dL * dRp;
                  if (emu_stage1 && dL >= emu_minM1 && dR >= emu_minK1 && dR <= 16384 && (int64_t)r.n * dRp >= emu_minN1) {
                    const int64_t kpad = (dR + 31) / 32 * 32, nlines = (int64_t)r.n * dRp;
                    const bool s1new = emu_s1new && kpad / 32 <= s1_kres;
                    std::vector<int> &pun = s1new ? punit32 : punit;
                    const int64_t prow = s1new ? 32 : 64;
                    if (pun[bi] < 0) {
                      pun[bi] = (int)P.sliceP.size();
                      EmuSliceDesc d{};
                      d.src = mkref(B_PSI_IN, b.off); d.lstride = 1; d.linestride = dR;
                      d.n_members = 1; d.dl = d.dlpad = (int32_t)dR; d.lines = (int32_t)dL; d.ld = kpad; d.tile_rows = prow;
                      d.out_off = P.emuP_bytes; d.exp_off = P.expP_n;
                      P.emuP_bytes += (dL + prow - 1) / prow * prow * kpad;
                      P.expP_n += (dL + 3) / 4 * 4;                  // 16-byte aligned segments (k_emu_s1 loads int4)
                      P.sliceP.push_back(d);
                    }
                    auto key = std::make_tuple(ra, (int)g.dagR, r.n);
                    auto ru = runits.find(key);
                    if (ru == runits.end()) {
                      ru = runits.emplace(key, std::make_pair(P.emuR_bytes, P.expR_n)).first;
                      EmuSliceDesc d{};
                      d.n_members = 1; d.dl = d.dlpad = (int32_t)dR; d.ld = kpad; d.tile_rows = 128;
                      d.s1_layout = s1new ? 1 : 0;             // a unit has one K, hence one consumer kernel
                      d.out_off = P.emuR_bytes; d.exp_off = P.expR_n;
                      if (!g.dagR) {            // stored [member][r'][r]: the lines are contiguous rows
                        d.src = ra; d.lstride = 1; d.linestride = dR; d.lines = (int32_t)nlines;
                        P.sliceR.push_back(d);
                      } else {                  // stored [member][r][r']: one descriptor per member
                        d.lstride = dRp; d.linestride = 1; d.lines = (int32_t)dRp;
                        for (int a = 0; a < r.n; ++a) {
                          d.src = ra + (int64_t)a * dR * dRp; d.line_base = (int32_t)(a * dRp);
                          P.sliceR.push_back(d);
                        }
                      }
                      P.emuR_bytes += (nlines + 127) / 128 * 128 * kpad; P.expR_n += nlines;
                    }
                    const EmuSliceDesc &dp = P.sliceP[pun[bi]];
                    EmuPass &E = P.emu[pass];
                    EmuSeg es{};
                    // A (128-row operand) = operator lines (member, r'): always full tiles; B (64 columns) = psi rows l
                    es.a_off = ru->second.first; es.ea_off = ru->second.second; es.b_off = dp.out_off; es.eb_off = dp.exp_off;
                    es.ksteps = (int32_t)(kpad / 32); es.alpha = 1.0;
                    EmuJob ej{};
                    ej.c = j1.c; ej.scale = j1.scale; ej.c_nhi = dL * dRp; ej.M = (int32_t)nlines; ej.N = (int32_t)dL;
                    ej.c_ld = (int32_t)dRp; ej.n1 = (int32_t)dRp; ej.rows_split = 1;
                    ej.seg_begin = (int32_t)E.segs1.size(); ej.seg_end = ej.seg_begin + 1;
                    ej.s1_new = s1new ? 1 : 0;
                    E.segs1.push_back(es);
                    if (!s1new)
                      for (int m0 = 0; m0 < ej.M; m0 += 128)
                        for (int n0 = 0; n0 < ej.N; n0 += 64) E.tiles1.push_back(EmuTile{(int32_t)E.jobs1.size(), m0, n0, 1});
                    ej1[ri] = (int)E.jobs1.size();
                    E.jobs1.push_back(ej);
                    P.flops_emu1 += 2 * dL * dR * r.n * dRp;
                  } else {
                    JobList &S1 = P.stage1v.back();
                    j1.seg_begin = (int32_t)S1.segs.size(); j1.seg_end = j1.seg_begin + 1;
                    S1.segs.push_back(s1);
                    S1.jobs.push_back(j1);
                  }
                  if (P.emu_mode && dlpad <= P.opt.emu_kpiece && (int64_t)r.n * dL >= emu_minK && dRp >= emu_minN && maxLp >= emu_minM) {
                    tuni[ri] = (int)P.emu[pass].sliceT.size();
                    int64_t qn = -1;
                    if (emu_bound) {           // line norms of the stacked right operators, once per bond
                      auto key = std::make_tuple(ra, (int)g.dagR, r.n, r.coef_off);
                      auto it = qnorms.find(key);
                      if (it == qnorms.end()) {
                        EmuNormDesc nd{};
                        nd.src = ra; nd.mstride = dRp * dR; nd.coef_off = r.coef_off; nd.out_off = P.emu_norm_elems;
                        if (!g.dagR) { nd.rstride = 1; nd.linestride = dR; } else { nd.rstride = dRp; nd.linestride = 1; }
                        nd.n_members = r.n; nd.dR = (int32_t)dR; nd.lines = (int32_t)dRp;
                        P.emu_norms.push_back(nd);
                        it = qnorms.emplace(key, P.emu_norm_elems).first;
                        P.emu_norm_elems += dRp;
                      }
                      qn = it->second;
                    }
                    for (int a0 = 0; a0 < r.n; a0 += per_piece) {
                      const int na = std::min(r.n - a0, per_piece);
                      EmuSliceDesc d{};
                      d.src = mkref(B_SCRATCH, toff[ri] + (int64_t)a0 * dL * dRp);
                      d.mstride = dL * dRp; d.lstride = dRp; d.linestride = 1;
                      d.n_members = na; d.dl = (int32_t)dL; d.dlpad = dlpad; d.lines = (int32_t)dRp;
                      d.ld = ((int64_t)na * dlpad + 31) / 32 * 32; d.out_off = emuT_cur; d.exp_off = expT_cur; d.tile_rows = 64;
                      d.qn_off = qn; d.psi_blk = (int32_t)bi; d.bound = qn >= 0;
                      if (ej1[ri] >= 0 && qn >= 0 && emu_fuse) {     // the emulated stage 1 writes these slices itself
                        d.bound = 2;
                        EmuJob &ej = P.emu[pass].jobs1[ej1[ri]];
                        if (a0 == 0) {
                          ej.fuse = 1; ej.t_out_off = d.out_off; ej.t_exp_off = d.exp_off; ej.qn_off = qn; ej.psi_blk = (int32_t)bi;
                          ej.per_piece = per_piece; ej.dlpad = dlpad; ej.ld_full = (int32_t)d.ld; ej.n_pieces = 0;
                          ej.piece_bytes = (d.lines + 63) / 64 * 64 * d.ld;
                        }
                        ej.ld_last = (int32_t)d.ld; ++ej.n_pieces;
                      }
                      emuT_cur += (d.lines + 63) / 64 * 64 * d.ld; expT_cur += d.lines;
                      P.emu[pass].sliceT.push_back(d);
                    }
                    P.emuT_bytes = std::max(P.emuT_bytes, emuT_cur);
                    P.expT_n = std::max(P.expT_n, expT_cur);
                  }
                  P.falg += 2 * dL * dR * r.n * dRp;
                  P.flops1 += 2 * dL * dR * r.n * dRp;
                  P.tab_falg_blocks[bo] += 2 * dL * dR * r.n * dRp;
                }
                P.falg += 2 * dLp * r.n * dL * dRp;
                P.flops2 += 2 * dLp * r.n * dL * dRp;
                P.tab_falg_blocks[bo] += 2 * dLp * r.n * dL * dRp;
                if (tuni[ri] >= 0 && dLp >= emu_minM) {     // emulated: one EmuSeg per member piece
                  auto key = std::make_tuple(la, (int)g.dagL, r.n);
                  auto lu = lunits.find(key);
                  if (lu == lunits.end()) {
                    lu = lunits.emplace(key, (int)P.sliceL.size()).first;
                    for (int a0 = 0; a0 < r.n; a0 += per_piece) {
                      const int na = std::min(r.n - a0, per_piece);
                      EmuSliceDesc d{};
                      d.src = la + (int64_t)a0 * dLp * dL;
                      d.mstride = dLp * dL;
                      if (!g.dagL) { d.lstride = 1; d.linestride = dL; } else { d.lstride = dLp; d.linestride = 1; }
                      d.n_members = na; d.dl = (int32_t)dL; d.dlpad = dlpad; d.lines = (int32_t)dLp;
                      d.ld = ((int64_t)na * dlpad + 31) / 32 * 32; d.out_off = P.emuL_bytes; d.exp_off = P.expL_n; d.tile_rows = 128;
                      P.emuL_bytes += (d.lines + 127) / 128 * 128 * d.ld; P.expL_n += d.lines;
                      P.sliceL.push_back(d);
                    }
                  }
                  int pc = 0;
                  for (int a0 = 0; a0 < r.n; a0 += per_piece, ++pc) {
                    const EmuSliceDesc &dl_ = P.sliceL[lu->second + pc], &dt = P.emu[tpass[ri]].sliceT[tuni[ri] + pc];
                    EmuSeg es{};
                    es.a_off = dl_.out_off; es.ea_off = dl_.exp_off;
                    es.b_off = dt.out_off; es.eb_off = dt.exp_off;
                    es.ksteps = (int32_t)(dl_.ld / 32); es.alpha = G;
                    esegs2[bo].push_back(es); epass2[bo].push_back(tpass[ri]);
                  }
                  P.flops_emu += 2 * dLp * r.n * dL * dRp;
                  continue;
                }
                // stage 2 segment (FP64): it reads T, so an emulated stage 1 must keep the FP64 copy
                if (ej1[ri] >= 0) P.emu[tpass[ri]].jobs1[ej1[ri]].write_fp64 = 1;
                sg.a = la; sg.K = (int32_t)(r.n * dL); sg.alpha = G;
                if (!g.dagL) { sg.a_ms = (int32_t)dL; sg.a_kn1 = (int32_t)dL; sg.a_klo = 1; sg.a_khi = dLp * dL; }
                else { sg.a_ms = 1; sg.a_kn1 = FLAT; sg.a_klo = (int32_t)dLp; sg.a_khi = 0; }
                sg.b = mkref(B_SCRATCH, toff[ri]); sg.b_ks = (int32_t)dRp; sg.b_nlo = 1; sg.b_nhi = 0;
                segs2[bo].push_back(sg); segn2[bo].push_back(r.n); segp2[bo].push_back(tpass[ri]);
              }
            }
        }
      }
    }
  }
  P.scratch_elems = max_scratch;
  const int n_pass = pass + 1;
  P.stage2v.assign(n_pass, JobList());
  // Stage-2 jobs, split along K into chunks of about equal work (segments are cut at operator-member
  // boundaries); a block with more than one chunk accumulates through B_PARTIAL and a fixed-order
  // reduction, so the result stays deterministic.
  int64_t tile_iters = 0;
  for (size_t bi = 0; bi < P.psi.size(); ++bi) {
    const PsiBlock &b = P.psi[bi];
    int64_t it = 0;
    for (const SegDesc &sg : segs2[bi]) it += (sg.K + 15) / 16;
    tile_iters += it * ((b.dL + BM - 1) / BM) * ((b.dR + BN - 1) / BN);
  }
  const int64_t target = std::max<int64_t>(24, tile_iters / (148 * 16));
  int64_t emu_iters = 0;
  for (size_t bi = 0; bi < P.psi.size(); ++bi) {
    int64_t ks = 0;
    for (const EmuSeg &es : esegs2[bi]) ks += es.ksteps;
    emu_iters += ks * ((P.psi[bi].dL + 127) / 128) * ((P.psi[bi].dR + 63) / 64);
  }
  const int64_t emu_target = std::max<int64_t>(64, emu_iters / (148 * 8));
  for (size_t bi = 0; bi < P.psi.size(); ++bi) {
    const PsiBlock &b = P.psi[bi];
    std::vector<SegDesc> pieces;
    std::vector<int> ppass;
    std::vector<size_t> order(segs2[bi].size());
    for (size_t i = 0; i < order.size(); ++i) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](size_t x, size_t y) { return segp2[bi][x] < segp2[bi][y]; });
    for (size_t si : order) {
      const SegDesc &sg = segs2[bi][si];
      const int n = segn2[bi][si], kper = sg.K / n;
      int per = (int)std::max<int64_t>(1, target * 16 / kper);
      for (int a0 = 0; a0 < n; a0 += per) {
        int a1 = std::min(n, a0 + per);
        SegDesc q = sg;
        q.K = (a1 - a0) * kper;
        q.a += (int64_t)a0 * (sg.a_kn1 != FLAT ? sg.a_khi : (int64_t)kper * sg.a_klo);
        q.b += (int64_t)a0 * kper * sg.b_ks;
        pieces.push_back(q);
        ppass.push_back(segp2[bi][si]);
      }
    }
    std::vector<std::pair<int, int>> chunks;   // [begin, end) over pieces
    int64_t acc_it = 0; int begin = 0;
    for (int pi = 0; pi < (int)pieces.size(); ++pi) {
      int64_t it = (pieces[pi].K + 15) / 16;
      if (pi > begin && (acc_it + it > target || ppass[pi] != ppass[begin])) { chunks.push_back({begin, pi}); begin = pi; acc_it = 0; }
      acc_it += it;
    }
    if (begin < (int)pieces.size() || esegs2[bi].empty()) chunks.push_back({begin, (int)pieces.size()});
    // emulated chunks: [begin, end) over the pass-sorted EmuSegs of this block
    std::vector<size_t> eorder(esegs2[bi].size());
    for (size_t i = 0; i < eorder.size(); ++i) eorder[i] = i;
    std::stable_sort(eorder.begin(), eorder.end(), [&](size_t x, size_t y) { return epass2[bi][x] < epass2[bi][y]; });
    std::vector<std::pair<int, int>> echunks;
    {
      int64_t acc = 0; int eb = 0;
      for (int ei = 0; ei < (int)eorder.size(); ++ei) {
        const int64_t ks = esegs2[bi][eorder[ei]].ksteps;
        if (ei > eb && (acc + ks > emu_target || epass2[bi][eorder[ei]] != epass2[bi][eorder[eb]])) { echunks.push_back({eb, ei}); eb = ei; acc = 0; }
        acc += ks;
      }
      if (!eorder.empty()) echunks.push_back({eb, (int)eorder.size()});
    }
    const int64_t mn = b.dL * b.dR;
    const size_t n_slots = chunks.size() + echunks.size();
    const bool direct = n_slots == 1;
    if (!direct) P.reduce.push_back(ReduceJob{b.off, P.partial_elems, (int32_t)mn, (int32_t)n_slots});
    for (size_t c = 0; c < chunks.size(); ++c) {
      JobDesc jd{};
      jd.c = direct ? mkref(B_PSI_OUT, b.off) : mkref(B_PARTIAL, P.partial_elems + (int64_t)c * mn);
      jd.scale = -1;
      jd.M = (int32_t)b.dL; jd.N = (int32_t)b.dR; jd.c_ms = (int32_t)b.dR; jd.n1 = FLAT; jd.c_nlo = 1; jd.c_nhi = 0;
      JobList &S2 = P.stage2v[chunks[c].first < chunks[c].second ? ppass[chunks[c].first] : 0];
      jd.seg_begin = (int32_t)S2.segs.size();
      S2.segs.insert(S2.segs.end(), pieces.begin() + chunks[c].first, pieces.begin() + chunks[c].second);
      jd.seg_end = (int32_t)S2.segs.size();
      S2.jobs.push_back(jd);
    }
    for (size_t c = 0; c < echunks.size(); ++c) {
      EmuPass &E = P.emu[epass2[bi][eorder[echunks[c].first]]];
      EmuJob ej{};
      ej.c = direct ? mkref(B_PSI_OUT, b.off) : mkref(B_PARTIAL, P.partial_elems + (int64_t)(chunks.size() + c) * mn);
      ej.M = (int32_t)b.dL; ej.N = (int32_t)b.dR; ej.c_ld = (int32_t)b.dR; ej.scale = -1; ej.n1 = FLAT; ej.c_nhi = 0;
      ej.seg_begin = (int32_t)E.segs.size();
      for (int ei = echunks[c].first; ei < echunks[c].second; ++ei) E.segs.push_back(esegs2[bi][eorder[ei]]);
      ej.seg_end = (int32_t)E.segs.size();
      for (int m0 = 0; m0 < ej.M; m0 += 128)
        for (int n0 = 0; n0 < ej.N; n0 += 64) E.tiles.push_back(EmuTile{(int32_t)E.jobs.size(), m0, n0, 1});
      E.jobs.push_back(ej);
    }
    if (!direct) P.partial_elems += (int64_t)n_slots * mn;
    DiagJob dj{b.off, (int32_t)b.dL, (int32_t)b.dR, (int32_t)P.diag_terms.size(), 0};
    P.diag_terms.insert(P.diag_terms.end(), diag[bi].begin(), diag[bi].end());
    dj.t_end = (int32_t)P.diag_terms.size();
    P.diag_jobs.push_back(dj);
  }
  int64_t nj1 = 0, ns1 = 0, nj2 = 0, ns2 = 0, nt1 = 0, nt2 = 0;
  for (int p = 0; p < n_pass; ++p) {
    make_tiles(P.stage1v[p], BM, BN, STRIP);
    make_tiles(P.stage2v[p], BM, BN, 1);
    nj1 += P.stage1v[p].jobs.size(); ns1 += P.stage1v[p].segs.size(); nt1 += P.stage1v[p].tiles.size();
    nj2 += P.stage2v[p].jobs.size(); ns2 += P.stage2v[p].segs.size(); nt2 += P.stage2v[p].tiles.size();
  }
  // heaviest tiles first: the INT8 launch of a pass has only a few CTAs per SM
  for (EmuPass &E : P.emu) {
    std::vector<int64_t> work(E.jobs.size(), 0);
    for (size_t j = 0; j < E.jobs.size(); ++j)
      for (int sgi = E.jobs[j].seg_begin; sgi < E.jobs[j].seg_end; ++sgi) work[j] += E.segs[sgi].ksteps + 2;
    std::stable_sort(E.tiles.begin(), E.tiles.end(), [&](const EmuTile &x, const EmuTile &y) { return work[x.job] > work[y.job]; });
  }
  // work items of the second-generation stage-1 kernel: jobs grouped by the right-operator unit they read
  for (EmuPass &E : P.emu) {
    std::map<int64_t, std::vector<int>> by_unit;
    for (size_t j = 0; j < E.jobs1.size(); ++j)
      if (E.jobs1[j].s1_new) by_unit[E.segs1[E.jobs1[j].seg_begin].a_off].push_back((int)j);
    for (auto &u : by_unit) {
      const EmuSeg &s0 = E.segs1[E.jobs1[u.second[0]].seg_begin];
      const int32_t M = E.jobs1[u.second[0]].M;
      const int32_t nt_begin = (int32_t)E.ntiles1.size();
      for (int j : u.second) {
        const EmuJob &jb = E.jobs1[j];
        const EmuSeg &sg = E.segs1[jb.seg_begin];
        if (jb.M != M || sg.ksteps != s0.ksteps || sg.ea_off != s0.ea_off) throw std::logic_error("stage-1 unit shared by unlike jobs");
        for (int n0 = 0; n0 < jb.N; n0 += 32)
          E.ntiles1.push_back(EmuS1Tile{sg.b_off + (int64_t)(n0 / 32) * sg.ksteps * 1024, j, n0, (int32_t)sg.eb_off, 0});
      }
      const int32_t nt_end = (int32_t)E.ntiles1.size();
      for (int m0 = 0; m0 < M; m0 += 128)
        E.items1.push_back(EmuS1Item{s0.a_off + (int64_t)(m0 / 128) * s0.ksteps * 4096, (int32_t)s0.ea_off, s0.ksteps, m0, M,
                                     nt_begin, nt_end, E.jobs1[u.second[0]].n1, 0});
    }
  }
  if (P.opt.debug) {          // what stays on the FP64 lists of stage 2, by the reason it stayed
    int64_t f_one = 0, f_k = 0, f_m = 0, f_n = 0, n_one = 0, n_k = 0, n_m = 0, n_n = 0, it_all = 0;
    for (size_t p = 0; p < P.stage2v.size(); ++p)
      for (const JobDesc &jd : P.stage2v[p].jobs)
        for (int si = jd.seg_begin; si < jd.seg_end; ++si) {
          const SegDesc &sg = P.stage2v[p].segs[si];
          const int64_t fl = 2ll * jd.M * jd.N * sg.K;
          it_all += (int64_t)((jd.M + BM - 1) / BM) * ((jd.N + BN - 1) / BN) * ((sg.K + 15) / 16);
          if (jd.M < emu_minM) { f_m += fl; ++n_m; }
          else if (jd.N < P.opt.emu_minn) { f_n += fl; ++n_n; }
          else if (sg.K < P.opt.emu_mink) { f_k += fl; ++n_k; }
          else { f_one += fl; ++n_one; }
        }
    fprintf(stderr, "[dmrg] FP64 stage-2 segments: d_L' small %lld (%.3g flop), d_R' small %lld (%.3g), K small %lld (%.3g), other (one-sided, pieces) %lld (%.3g); tile k-iterations %lld\n",
            (long long)n_m, (double)f_m, (long long)n_n, (double)f_n, (long long)n_k, (double)f_k, (long long)n_one, (double)f_one, (long long)it_all);
  }
  if (P.opt.debug)
    for (const EmuPass &E : P.emu) {
      int64_t nt = 0, ks = 0;
      for (const EmuS1Item &it : E.items1) { nt += it.nt_end - it.nt_begin; ks += (int64_t)(it.nt_end - it.nt_begin) * it.ksteps; }
      fprintf(stderr, "[dmrg] pass: s1 items %zu, n-tiles listed %zu, tile visits %lld (avg %.1f per item, %.2f k steps per tile), old-kernel tiles %zu\n",
              E.items1.size(), E.ntiles1.size(), (long long)nt, E.items1.empty() ? 0.0 : (double)nt / E.items1.size(),
              nt ? (double)ks / nt : 0.0, E.tiles1.size());
    }
  int64_t n_eseg = 0, n_etile = 0;
  for (const EmuPass &E : P.emu) { n_eseg += (int64_t)E.segs.size(); n_etile += (int64_t)E.tiles.size(); }
  for (const Group &g : P.groups) {
    int64_t n = 0;
    for (auto &r : g.runs) n += r.n;
    int64_t row[9] = {g.s1p, g.s1, g.s2p, g.s2, Lb.classes[g.clsL].kind, g.dagL, Rb.classes[g.clsR].kind,
                      g.dagR, n};
    P.tab_groups.insert(P.tab_groups.end(), row, row + 9);
  }
  // every emulated descriptor must stay inside its slice buffer (the kernels fetch whole tiles by bulk copy)
  for (size_t p = 0; p < P.emu.size(); ++p) {
    const EmuPass &E = P.emu[p];
    for (int stage = 1; stage <= 2; ++stage) {
      const auto &jobs = stage == 1 ? E.jobs1 : E.jobs;
      const auto &sgs = stage == 1 ? E.segs1 : E.segs;
      const int64_t a_cap = stage == 1 ? P.emuR_bytes : P.emuL_bytes, b_cap = stage == 1 ? P.emuP_bytes : P.emuT_bytes;
      for (const EmuJob &j : jobs) {
        const int64_t brow = (stage == 1 && j.s1_new) ? 32 : 64;          // rows of a B tile
        const int64_t tm = (j.M + 127) / 128, tn = (j.N + brow - 1) / brow;
        for (int sgi = j.seg_begin; sgi < j.seg_end; ++sgi) {
          const EmuSeg &sg = sgs[sgi];
          if (sg.ksteps < 1 || sg.ksteps > 512 || sg.a_off < 0 || sg.b_off < 0 ||
              sg.a_off + tm * sg.ksteps * 4096 > a_cap || sg.b_off + tn * sg.ksteps * (brow * 32) > b_cap)
            throw std::logic_error("emulated segment outside its slice buffer");
        }
        if (j.fuse && (j.t_out_off < 0 || j.t_out_off + (int64_t)(j.n_pieces - 1) * j.piece_bytes +
                                              (int64_t)(j.n1 + 63) / 64 * 64 * j.ld_last > P.emuT_bytes))
          throw std::logic_error("fused T unit outside the T slice buffer");
      }
    }
  }
  P.tab_opL = op_block_table(Lb);
  P.tab_opR = op_block_table(Rb);
  P.tab_counts = {nj1, ns1, nj2, ns2, nt1, nt2, P.scratch_elems, Lb.elems, Rb.elems, P.derL_elems, P.derR_elems,
                  P.flops1, P.flops2, P.partial_elems, (int64_t)n_pass, P.flops_emu, n_eseg, n_etile, P.flops_emu1};
}

}  // namespace dmrg
