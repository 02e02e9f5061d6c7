// H_eff plan for both symmetries: psi block table, reduction of the symbolic term list into
// class-stacked groups with derived (integral-contracted) operators, geometry factors (fermion
// signs for U(1)xU(1), 6j/9j recoupling for SU(2)), and the stage-1 /
// stage-2 / diagonal descriptors (rows a2, a3, a5, a6, a7 of section 8(a)).
#include <algorithm>
#include <cmath>
#include <stdexcept>

#include "internal.h"

namespace dmrg {

namespace {
struct GKey {
  int clsL, dagL, clsR, dagR, unit, k1, kk, k2;
  bool operator<(const GKey &o) const {
    return std::tie(clsL, dagL, clsR, dagR, unit, k1, kk, k2) <
           std::tie(o.clsL, o.dagL, o.clsR, o.dagR, o.unit, o.k1, o.kk, o.k2);
  }
};
struct Entry { Sym L, R; double c; };
inline bool tri2(int a, int b, int c) { return c >= std::abs(a - b) && c <= a + b && ((a + b + c) % 2) == 0; }
// <bra||T~||ket> = tilde_factor * <ket||T||bra>   (doubled spins S_bra, S_ket, rank k)
inline double tilde_factor(int S_bra, int S_ket, int k2) {
  int e = (S_ket - S_bra + k2) / 2;
  return ((e & 1) ? -1.0 : 1.0) * std::sqrt((S_ket + 1.0) / (S_bra + 1.0));
}
}  // namespace

void build_heff_plan(HeffPlan &P, const Integrals &ints, const BlockState &Lb, const BlockState &Rb,
                     int site1, int site2, int N, int twoS, int BM, int BN, int64_t scratch_budget, bool emu, bool tf32,
                     int kappa, const PlanOptions *opt) {
  P = HeffPlan();
  if (opt) P.opt = *opt;
  P.scratch_budget = scratch_budget;
  P.emu_mode = emu;
  P.emu_tf32 = tf32;
  P.kappa = kappa;
  const int sym = Lb.sym, ns = n_site_states(sym);
  P.resL.ints = &ints; P.resL.blk = &Lb;
  P.resR.ints = &ints; P.resR.blk = &Rb;
  // --- psi blocks, lexicographic (iL, s1, SA, s2, iR, SB)
  for (int iL = 0; iL < (int)Lb.tab.sec.size(); ++iL)
    for (int s1 = 0; s1 < ns; ++s1)
      for (int SA : fuse_S(sym, Lb.tab.sec[iL].S, s1))
        for (int s2 = 0; s2 < ns; ++s2)
          for (int iR = 0; iR < (int)Rb.tab.sec.size(); ++iR) {
            const Sector &qL = Lb.tab.sec[iL], &qR = Rb.tab.sec[iR];
            if (qL.N + site_N(sym, s1) + site_N(sym, s2) + qR.N != N) continue;
            for (int SB : fuse_S(sym, qR.S, s2)) {
              if (sym == 0 ? (SA + SB != twoS) : !tri2(SA, SB, twoS)) continue;
              PsiBlock pb{iL, s1, SA, s2, iR, SB, qL.dim, qR.dim, P.psi_len};
              P.psi_index[std::make_tuple(iL, s1, SA, s2, iR, SB)] = (int)P.psi.size();
              P.psi.push_back(pb);
              P.psi_len += pb.dL * pb.dR;
            }
          }
  for (auto &pb : P.psi) {
    if (sym == 0) {
      int64_t row[7] = {pb.iL, pb.s1, pb.s2, pb.iR, pb.dL, pb.dR, pb.off};
      P.tab_psi.insert(P.tab_psi.end(), row, row + 7);
    } else {
      int64_t row[9] = {pb.iL, pb.s1, pb.SA, pb.s2, pb.iR, pb.SB, pb.dL, pb.dR, pb.off};
      P.tab_psi.insert(P.tab_psi.end(), row, row + 9);
    }
  }
  // --- symbolic terms, grouped by (class, dagger/tilde) of both sides, the site unit and the ranks
  std::vector<HTerm> terms = sym == 0 ? heff_terms(ints, Lb.orbs, site1, site2, Rb.orbs)
                                      : heff_terms_su2(ints, Lb.orbs, site1, site2, Rb.orbs);
  std::map<GKey, std::vector<Entry>> groups;
  for (const HTerm &t : terms) {
    int cl, dl, cr, dr;
    if (!P.resL.flat(t.L, &cl, &dl, nullptr, nullptr)) continue;
    if (!P.resR.flat(t.R, &cr, &dr, nullptr, nullptr)) continue;
    int unit = ((t.s1p * 4 + t.s1) * 4 + t.s2p) * 4 + t.s2;
    groups[GKey{cl, dl, cr, dr, unit, t.k1, t.kk, t.k2}].push_back({t.L, t.R, t.c});
  }
  int64_t run_coef_elems = 0;
  for (auto &ge : groups) {
    const GKey &k = ge.first;
    // merge duplicate (L, R) pairs, then pair up or contract
    std::map<std::pair<Sym, Sym>, double> merged;
    for (auto &e : ge.second) merged[{e.L, e.R}] += e.c;
    std::map<Sym, std::vector<std::pair<Sym, double>>> byL, byR;
    for (auto &m : merged) {
      if (m.second == 0.0) continue;
      byL[m.first.first].push_back({m.first.second, m.second});
      byR[m.first.second].push_back({m.first.first, m.second});
    }
    if (byL.empty()) continue;
    bool one2one = true;
    for (auto &x : byL) if (x.second.size() != 1) one2one = false;
    for (auto &x : byR) if (x.second.size() != 1) one2one = false;
    struct Alpha { OpRef L, R; double c; };
    std::vector<Alpha> al;
    int dagtmp;
    if (one2one) {
      for (auto &x : byL)
        al.push_back({P.resL.resolve(x.first, &dagtmp), P.resR.resolve(x.second[0].first, &dagtmp),
                      x.second[0].second});
    } else if (byL.size() >= byR.size()) {   // contract the left side onto each right symbol
      for (auto &x : byR) {
        std::vector<double> w(Lb.classes[k.clsL].n(), 0.0), wa;
        for (auto &a : x.second) {
          int c_, d_;
          P.resL.flat(a.first, &c_, &d_, &wa, nullptr);
          for (size_t i = 0; i < w.size(); ++i) w[i] += a.second * wa[i];
        }
        al.push_back({P.resL.resolve_weights(k.clsL, w), P.resR.resolve(x.first, &dagtmp), 1.0});
      }
    } else {
      for (auto &x : byL) {
        std::vector<double> w(Rb.classes[k.clsR].n(), 0.0), wa;
        for (auto &a : x.second) {
          int c_, d_;
          P.resR.flat(a.first, &c_, &d_, &wa, nullptr);
          for (size_t i = 0; i < w.size(); ++i) w[i] += a.second * wa[i];
        }
        al.push_back({P.resL.resolve(x.first, &dagtmp), P.resR.resolve_weights(k.clsR, w), 1.0});
      }
    }
    Group g;
    g.s2 = k.unit % 4; g.s2p = (k.unit / 4) % 4; g.s1 = (k.unit / 16) % 4; g.s1p = k.unit / 64;
    g.clsL = k.clsL; g.dagL = k.dagL; g.clsR = k.clsR; g.dagR = k.dagR;
    g.k1 = k.k1; g.kk = k.kk; g.k2 = k.k2;
    g.dqL = Lb.classes[k.clsL].dq; g.dqR = Rb.classes[k.clsR].dq;
    if (k.dagL) g.dqL.dN = -g.dqL.dN;
    if (k.dagR) g.dqR.dN = -g.dqR.dN;
    if (sym == 0) { if (k.dagL) g.dqL.dS = -g.dqL.dS; if (k.dagR) g.dqR.dS = -g.dqR.dS; }
    for (size_t a = 0; a < al.size(); ++a) {
      if (a > 0 && consecutive(al[a - 1].L, al[a].L) && consecutive(al[a - 1].R, al[a].R)) {
        g.runs.back().n++;
        g.runs.back().c.push_back(al[a].c);
      } else {
        g.runs.push_back(Run{al[a].L, al[a].R, 1, 0, {al[a].c}});
      }
    }
    for (Run &r : g.runs) { r.coef_off = run_coef_elems; run_coef_elems += r.n; }
    P.groups.push_back(std::move(g));
  }
  // --- derived operators (a3) and the coefficient buffer: [W_L][W_R][run coefficients]
  int64_t coefL = 0, coefR = 0;
  P.derL_elems = P.resL.finalize(&coefL);
  P.derR_elems = P.resR.finalize(&coefR);
  P.resL.coef_data(P.coef);
  P.resR.coef_data(P.coef);
  const int64_t run_base = coefL + coefR;
  for (Group &g : P.groups)
    for (Run &r : g.runs) {
      r.coef_off += run_base;
      for (double c : r.c) P.coef.push_back(c);
    }
  P.resL.contraction_jobs(P.contractL, B_OPS_L, B_DER_L, 0);
  P.resR.contraction_jobs(P.contractR, B_OPS_R, B_DER_R, coefL);
  make_tiles(P.contractL, BM, BN, STRIP);
  make_tiles(P.contractR, BM, BN, STRIP);
  // In the tensor-core modes the FP64 lists of the two stages hold only the remainder (one-sided terms and segments below
  // the size thresholds): small blocks, which waste less on the smallest tile (configs[2]: 7.2 -> 5.5 ms, configs[4]:
  // 688 -> 511 ms per apply with 32 instead of 64); the option `tile` still overrides.
  const int st = (P.emu_mode && P.opt.tile == 0) ? 32 : BM;
  build_heff_jobs(P, Lb, Rb, N, twoS, st, P.emu_mode && P.opt.tile == 0 ? 32 : BN);
}

}  // namespace dmrg
