// Host-side planning: symmetry tables, operator layouts, reduction of the symbolic term
// lists into class-stacked groups with derived (integral-contracted) operators, and the
// flat job/segment descriptors executed by the device kernels.
// SURVEY.md section 8(a) rows a2, a3 (plans), a5, a6, a7, a9 (descriptors); section 7
// "class-stacked layout".
#include "internal.h"

#include <algorithm>
#include <cmath>
#include <stdexcept>

namespace dmrg {

static const int32_t FLAT = 1 << 30;   // n1 / kn1 value of a single-level index
static const int STRIP = 8;            // n-tiles per CTA for the short-K lists (stage 1, rotation 1, contraction)

BondTable make_table(const int64_t *rows, int64_t n) {
  BondTable t;
  int64_t off = 0;
  for (int64_t r = 0; r < n; ++r) {
    Sector s{(int)rows[4 * r], (int)rows[4 * r + 1], rows[4 * r + 2], off};
    if (s.dim <= 0) throw std::invalid_argument("bond table: non-positive sector dimension");
    if (t.index.count({s.N, s.S})) throw std::invalid_argument("bond table: duplicate sector");
    if (!t.sec.empty()) {
      const Sector &p = t.sec.back();
      if (std::make_pair(p.N, p.S) >= std::make_pair(s.N, s.S))
        throw std::invalid_argument("bond table: rows not sorted by (N, twoS)");
    }
    t.index[{s.N, s.S}] = (int)t.sec.size();
    t.sec.push_back(s);
    off += s.dim;
  }
  t.total = off;
  return t;
}

std::vector<IsoBlock> iso_blocks(const BondTable &prev, const BondTable &next, int64_t *total) {
  std::vector<IsoBlock> out;
  int64_t off = 0;
  for (int ip = 0; ip < (int)prev.sec.size(); ++ip)
    for (int s = 0; s < 4; ++s) {
      int in = next.find(prev.sec[ip].N + SITE_N[s], prev.sec[ip].S + SITE_S[s]);
      if (in < 0) continue;
      IsoBlock b{ip, s, in, prev.sec[ip].dim, next.sec[in].dim, off};
      off += b.rows * b.cols;
      out.push_back(b);
    }
  if (total) *total = off;
  return out;
}

// ----------------------------------------------------------------------------- layouts
void layout_block(BlockState &b, int L) {
  b.classes.clear();
  b.class_index.clear();
  std::vector<char> in(2 * L, 0);
  for (int i : b.orbs) in[i] = 1;
  auto cls = [&](int kind, DQ dq) -> OpClass & {
    auto key = std::make_tuple(kind, dq.dN, dq.dS);
    auto it = b.class_index.find(key);
    if (it == b.class_index.end()) {
      b.class_index[key] = (int)b.classes.size();
      b.classes.push_back(OpClass{kind, dq, {}, {}, {}, {}});
      return b.classes.back();
    }
    return b.classes[it->second];
  };
  auto add = [&](int kind, int i, int k) {
    Sym s{kind, 0, i, k};
    OpClass &c = cls(kind, sym_dq(s));
    c.member_index[{i, k}] = c.n();
    c.members.push_back({i, k});
  };
  add(K_I, -1, -1);
  if (!b.orbs.empty()) {
    add(K_H, -1, -1);
    for (int i : b.orbs) add(K_C, i, -1);
    for (int x = 0; x < 2 * L; ++x) if (!in[x]) add(K_S, x, -1);
    for (size_t a = 0; a < b.orbs.size(); ++a)
      for (size_t c = a + 1; c < b.orbs.size(); ++c) add(K_A, b.orbs[a], b.orbs[c]);
    for (int i : b.orbs) for (int l : b.orbs) add(K_B, i, l);
  }
  int64_t off = 0;
  for (OpClass &c : b.classes) {
    for (int ket = 0; ket < (int)b.tab.sec.size(); ++ket) {
      int bra = b.tab.find(b.tab.sec[ket].N + c.dq.dN, b.tab.sec[ket].S + c.dq.dS);
      if (bra < 0) continue;
      c.blocks.push_back({bra, ket, 0});
    }
    std::sort(c.blocks.begin(), c.blocks.end(), [](const OpBlock &x, const OpBlock &y) {
      return x.bra != y.bra ? x.bra < y.bra : x.ket < y.ket; });
    for (size_t i = 0; i < c.blocks.size(); ++i) {
      OpBlock &ob = c.blocks[i];
      ob.off = off;
      off += (int64_t)c.n() * b.tab.sec[ob.bra].dim * b.tab.sec[ob.ket].dim;
      c.block_index[{ob.bra, ob.ket}] = (int)i;
    }
  }
  b.elems = off;
}

std::vector<OpKey> block_targets(const BlockState &b) {
  std::vector<OpKey> t;
  for (const OpClass &c : b.classes)
    for (auto &m : c.members) t.push_back({c.kind, m.first, m.second});
  return t;
}

std::vector<int64_t> op_block_table(const BlockState &b) {
  std::vector<int64_t> t;
  for (const OpClass &c : b.classes)
    for (const OpBlock &ob : c.blocks) {
      int64_t row[7] = {c.kind, c.dq.dN, c.dq.dS, c.n(), ob.bra, ob.ket, ob.off};
      t.insert(t.end(), row, row + 7);
    }
  return t;
}

void make_tiles(JobList &jl, int BM, int BN, int strip) {
  // One CTA per (job, m-tile, strip of up to `strip` consecutive n-tiles); heaviest first, so the
  // hardware block scheduler balances the load.  TileDesc.work carries the strip length to the device.
  jl.tiles.clear();
  jl.tile = BM;
  std::vector<std::pair<int64_t, TileDesc>> tmp;
  for (int j = 0; j < (int)jl.jobs.size(); ++j) {
    JobDesc &jd = jl.jobs[j];
    int64_t k = 0, iters = 0;
    for (int s = jd.seg_begin; s < jd.seg_end; ++s) { k += jl.segs[s].K; iters += (jl.segs[s].K + 15) / 16; }
    jd.n_iters = (int32_t)iters;
    for (int m0 = 0; m0 < jd.M; m0 += BM)
      for (int n0 = 0; n0 < jd.N; n0 += BN * strip) {
        int64_t mm = std::min(BM, jd.M - m0), nn = std::min(BN * strip, jd.N - n0);
        int cnt = (int)((nn + BN - 1) / BN);
        // work estimate in units of 8x8x4 MMA steps (what the FP64 tensor pipe executes)
        int64_t w = ((mm + 7) / 8) * ((nn + 7) / 8) * ((k + 3) / 4) + 16;
        tmp.push_back({w, TileDesc{j, m0, n0, cnt}});
      }
  }
  std::stable_sort(tmp.begin(), tmp.end(),
                   [](const std::pair<int64_t, TileDesc> &a, const std::pair<int64_t, TileDesc> &b) {
                     return a.first > b.first; });
  jl.tiles.reserve(tmp.size());
  for (auto &t : tmp) jl.tiles.push_back(t.second);
}

// ----------------------------------------------------------------------------- resolver
bool Resolver::flat(const Sym &s, int *cls, int *dag, std::vector<double> *w, int *single_idx) const {
  const BlockState &b = *blk;
  if (single_idx) *single_idx = -1;
  if (s.kind == K_P) {
    // P_ik = sum_{j<l in R} (v_ijkl - v_ilkj) (A_jl)+       (Appendix A2)
    int c = b.find_class(K_A, DQ{2, spin_of(s.i) + spin_of(s.k)});
    if (c < 0) return false;
    *cls = c; *dag = !s.dag;
    if (w) {
      const OpClass &oc = b.classes[c];
      w->assign(oc.n(), 0.0);
      for (int a = 0; a < oc.n(); ++a) {
        int j = oc.members[a].first, l = oc.members[a].second;
        (*w)[a] = ints->v(s.i, j, s.k, l) - ints->v(s.i, l, s.k, j);
      }
    }
    return true;
  }
  if (s.kind == K_Q) {
    // Q_il = sum_{k,j in R} (v_ilkj - v_ijkl) B_kj
    int c = b.find_class(K_B, DQ{0, spin_of(s.k) - spin_of(s.i)});
    if (c < 0) return false;
    *cls = c; *dag = 0;
    if (w) {
      const OpClass &oc = b.classes[c];
      w->assign(oc.n(), 0.0);
      for (int a = 0; a < oc.n(); ++a) {
        int k = oc.members[a].first, j = oc.members[a].second;
        (*w)[a] = ints->v(s.i, s.k, k, j) - ints->v(s.i, j, k, s.k);
      }
    }
    return true;
  }
  Sym u = s; u.dag = 0;
  int c = b.find_class(s.kind, sym_dq(u));
  if (c < 0) return false;
  const OpClass &oc = b.classes[c];
  auto it = oc.member_index.find({s.i, s.k});
  if (it == oc.member_index.end()) return false;
  *cls = c; *dag = s.dag;
  if (single_idx) *single_idx = it->second;
  if (w) { w->assign(oc.n(), 0.0); (*w)[it->second] = 1.0; }
  return true;
}

OpRef Resolver::resolve_weights(int cls, const std::vector<double> &w) {
  auto it = derived_of_class.find(cls);
  int d;
  if (it == derived_of_class.end()) {
    d = (int)derived.size();
    derived_of_class[cls] = d;
    derived.push_back(DerivedClass{cls, {}, {}, {}, 0});
  } else d = it->second;
  DerivedClass &dc = derived[d];
  auto f = dc.dedupe.find(w);
  if (f != dc.dedupe.end()) return OpRef{1, d, f->second};
  int idx = (int)dc.weights.size();
  dc.weights.push_back(w);
  dc.dedupe[w] = idx;
  return OpRef{1, d, idx};
}

OpRef Resolver::resolve(const Sym &s, int *dag) {
  int cls, single;
  std::vector<double> w;
  bool stored = (s.kind != K_P && s.kind != K_Q);
  if (!flat(s, &cls, dag, stored ? nullptr : &w, &single)) throw std::logic_error("unresolvable symbol");
  if (stored) return OpRef{0, cls, single};
  return resolve_weights(cls, w);
}

int64_t Resolver::finalize(int64_t *coef_elems) {
  int64_t off = 0, co = 0;
  for (DerivedClass &dc : derived) {
    const OpClass &oc = blk->classes[dc.cls];
    dc.block_off.clear();
    for (const OpBlock &ob : oc.blocks) {
      dc.block_off.push_back(off);
      off += (int64_t)dc.weights.size() * blk->tab.sec[ob.bra].dim * blk->tab.sec[ob.ket].dim;
    }
    dc.coef_off = co;
    co += (int64_t)dc.weights.size() * oc.n();
  }
  if (coef_elems) *coef_elems = co;
  return off;
}

void Resolver::coef_data(std::vector<double> &out) const {
  for (const DerivedClass &dc : derived)
    for (auto &row : dc.weights) out.insert(out.end(), row.begin(), row.end());
}

// a3: derived[beta][e] = sum_alpha W[beta][alpha] stored[alpha][e], one GEMM per sector pair.
void Resolver::contraction_jobs(JobList &jl, int buf_ops, int buf_der, int64_t coef_base) const {
  for (const DerivedClass &dc : derived) {
    const OpClass &oc = blk->classes[dc.cls];
    int nd = (int)dc.weights.size(), nm = oc.n();
    for (size_t bi = 0; bi < oc.blocks.size(); ++bi) {
      const OpBlock &ob = oc.blocks[bi];
      int64_t e = blk->tab.sec[ob.bra].dim * blk->tab.sec[ob.ket].dim;
      if (e > INT32_MAX) throw std::runtime_error("operator block too large");
      SegDesc sg{};
      sg.a = mkref(B_COEF, coef_base + dc.coef_off); sg.a_ms = nm; sg.a_kn1 = FLAT; sg.a_klo = 1; sg.a_khi = 0;
      sg.b = mkref(buf_ops, ob.off); sg.b_ks = (int32_t)e; sg.b_nlo = 1; sg.b_nhi = 0;
      sg.K = nm; sg.alpha = 1.0;
      JobDesc jd{};
      jd.c = mkref(buf_der, dc.block_off[bi]); jd.scale = -1;
      jd.M = nd; jd.N = (int32_t)e; jd.c_ms = (int32_t)e; jd.n1 = FLAT; jd.c_nlo = 1; jd.c_nhi = 0;
      jd.seg_begin = (int32_t)jl.segs.size(); jd.seg_end = jd.seg_begin + 1;
      jl.segs.push_back(sg);
      jl.jobs.push_back(jd);
      jl.flops += 2LL * nd * nm * e;
    }
  }
}

// address of member idx of operator `r` for the stored-orientation block (bra, ket)
static bool op_addr(const Resolver &res, const OpRef &r, int buf_ops, int buf_der, int bra, int ket,
                    ref_t *ref, int *cls_out) {
  const BlockState &b = *res.blk;
  int cls = r.derived ? res.derived[r.arr].cls : r.arr;
  const OpClass &oc = b.classes[cls];
  auto it = oc.block_index.find({bra, ket});
  if (it == oc.block_index.end()) return false;
  int64_t e = b.tab.sec[bra].dim * b.tab.sec[ket].dim;
  if (r.derived) *ref = mkref(buf_der, res.derived[r.arr].block_off[it->second] + (int64_t)r.idx * e);
  else *ref = mkref(buf_ops, oc.blocks[it->second].off + (int64_t)r.idx * e);
  if (cls_out) *cls_out = cls;
  return true;
}

static bool consecutive(const OpRef &a, const OpRef &b) {
  return a.derived == b.derived && a.arr == b.arr && b.idx == a.idx + 1;
}

// ----------------------------------------------------------------------------- H_eff plan
namespace {
struct GKey {
  int clsL, dagL, clsR, dagR, unit;
  bool operator<(const GKey &o) const {
    return std::tie(clsL, dagL, clsR, dagR, unit) < std::tie(o.clsL, o.dagL, o.clsR, o.dagR, o.unit);
  }
};
struct Entry { Sym L, R; double c; };
}  // namespace

void build_heff_plan(HeffPlan &P, const Integrals &ints, const BlockState &Lb, const BlockState &Rb,
                     int site1, int site2, int N, int twoS, int BM, int BN) {
  P = HeffPlan();
  P.resL.ints = &ints; P.resL.blk = &Lb;
  P.resR.ints = &ints; P.resR.blk = &Rb;
  // --- psi blocks, lexicographic (iL, s1, s2, iR)
  for (int iL = 0; iL < (int)Lb.tab.sec.size(); ++iL)
    for (int s1 = 0; s1 < 4; ++s1)
      for (int s2 = 0; s2 < 4; ++s2) {
        const Sector &q = Lb.tab.sec[iL];
        int iR = Rb.tab.find(N - q.N - SITE_N[s1] - SITE_N[s2], twoS - q.S - SITE_S[s1] - SITE_S[s2]);
        if (iR < 0) continue;
        PsiBlock pb{iL, s1, s2, iR, q.dim, Rb.tab.sec[iR].dim, P.psi_len};
        P.psi_index[std::make_tuple(iL, s1, s2, iR)] = (int)P.psi.size();
        P.psi.push_back(pb);
        P.psi_len += pb.dL * pb.dR;
      }
  for (auto &pb : P.psi) {
    int64_t row[7] = {pb.iL, pb.s1, pb.s2, pb.iR, pb.dL, pb.dR, pb.off};
    P.tab_psi.insert(P.tab_psi.end(), row, row + 7);
  }
  // --- symbolic terms, grouped by (class, dagger) of both sides and the site unit
  std::vector<HTerm> terms = heff_terms(ints, Lb.orbs, site1, site2, Rb.orbs);
  std::map<GKey, std::vector<Entry>> groups;
  for (const HTerm &t : terms) {
    int cl, dl, cr, dr;
    if (!P.resL.flat(t.L, &cl, &dl, nullptr, nullptr)) continue;
    if (!P.resR.flat(t.R, &cr, &dr, nullptr, nullptr)) continue;
    int unit = ((t.s1p * 4 + t.s1) * 4 + t.s2p) * 4 + t.s2;
    groups[GKey{cl, dl, cr, dr, unit}].push_back({t.L, t.R, t.c});
  }
  int64_t run_coef_elems = 0;
  for (auto &ge : groups) {
    const GKey &k = ge.first;
    std::vector<Entry> &es = ge.second;
    std::map<Sym, std::vector<std::pair<Sym, double>>> byL, byR;
    for (auto &e : es) { byL[e.L].push_back({e.R, e.c}); byR[e.R].push_back({e.L, e.c}); }
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
    g.dqL = Lb.classes[k.clsL].dq; g.dqR = Rb.classes[k.clsR].dq;
    if (k.dagL) g.dqL = DQ{-g.dqL.dN, -g.dqL.dS};
    if (k.dagR) g.dqR = DQ{-g.dqR.dN, -g.dqR.dS};
    for (size_t a = 0; a < al.size(); ++a) {
      if (a > 0 && consecutive(al[a - 1].L, al[a].L) && consecutive(al[a - 1].R, al[a].R)) {
        g.runs.back().n++;
        g.runs.back().c.push_back(al[a].c);
      } else {
        g.runs.push_back(Run{al[a].L, al[a].R, 1, 0, {al[a].c}});
      }
    }
    for (Run &r : g.runs) { r.coef_off = run_coef_elems; run_coef_elems += 2 * r.n; }
    P.groups.push_back(std::move(g));
  }
  // --- derived operators (a3) and the coefficient buffer: [W_L][W_R][run coefficients +-]
  int64_t coefL = 0, coefR = 0;
  P.derL_elems = P.resL.finalize(&coefL);
  P.derR_elems = P.resR.finalize(&coefR);
  P.resL.coef_data(P.coef);
  P.resR.coef_data(P.coef);
  int64_t run_base = coefL + coefR;
  for (Group &g : P.groups)
    for (Run &r : g.runs) {
      r.coef_off += run_base;
      for (double c : r.c) P.coef.push_back(c);
      for (double c : r.c) P.coef.push_back(-c);
    }
  P.resL.contraction_jobs(P.contractL, B_OPS_L, B_DER_L, 0);
  P.resR.contraction_jobs(P.contractR, B_OPS_R, B_DER_R, coefL);
  make_tiles(P.contractL, BM, BN, STRIP);
  make_tiles(P.contractR, BM, BN, STRIP);

  // --- stage 1 / stage 2 descriptors (a5, a6) and the diagonal terms (a7)
  std::vector<std::vector<SegDesc>> segs2(P.psi.size());
  std::vector<std::vector<int>> segn2(P.psi.size());   // members per stage-2 segment
  std::vector<std::vector<DiagTerm>> diag(P.psi.size());
  int64_t scratch = 0;
  P.tab_falg_blocks.assign(P.psi.size(), 0);
  for (const Group &g : P.groups) {
    int kindL = Lb.classes[g.clsL].kind, kindR = Rb.classes[g.clsR].kind;
    int pi1 = (SITE_N[g.s1p] - SITE_N[g.s1]) & 1, pi2 = (SITE_N[g.s2p] - SITE_N[g.s2]) & 1;
    int piR = g.dqR.dN & 1;
    for (size_t bi = 0; bi < P.psi.size(); ++bi) {
      const PsiBlock &b = P.psi[bi];
      if (b.s1 != g.s1 || b.s2 != g.s2) continue;
      const Sector &qL = Lb.tab.sec[b.iL], &qR = Rb.tab.sec[b.iR];
      int iLp = Lb.tab.find(qL.N + g.dqL.dN, qL.S + g.dqL.dS);
      int iRp = Rb.tab.find(qR.N + g.dqR.dN, qR.S + g.dqR.dS);
      if (iLp < 0 || iRp < 0) continue;
      auto po = P.psi_index.find(std::make_tuple(iLp, g.s1p, g.s2p, iRp));
      if (po == P.psi_index.end()) continue;
      const PsiBlock &bo = P.psi[po->second];
      // Appendix A5 sign: (-1)^{N_l(pi1+pi2+piR) + N_s1(pi2+piR) + N_s2 piR}
      int e = qL.N * (pi1 + pi2 + piR) + SITE_N[b.s1] * (pi2 + piR) + SITE_N[b.s2] * piR;
      double sgn = (e & 1) ? -1.0 : 1.0;
      int64_t dL = b.dL, dR = b.dR, dLp = bo.dL, dRp = bo.dR;
      // stored-orientation block labels of the two operators
      int lbra = g.dagL ? b.iL : iLp, lket = g.dagL ? iLp : b.iL;
      int rbra = g.dagR ? b.iR : iRp, rket = g.dagR ? iRp : b.iR;
      bool diagonal = (g.s1p == g.s1 && g.s2p == g.s2 && iLp == b.iL && iRp == b.iR);
      for (const Run &r : g.runs) {
        ref_t la, ra;
        if (!op_addr(P.resL, r.L, B_OPS_L, B_DER_L, lbra, lket, &la, nullptr)) continue;
        if (!op_addr(P.resR, r.R, B_OPS_R, B_DER_R, rbra, rket, &ra, nullptr)) continue;
        if (diagonal)
          for (int a = 0; a < r.n; ++a)
            diag[bi].push_back({la + a * dL * dL, ra + a * dR * dR, (int32_t)(dL + 1), (int32_t)(dR + 1),
                                sgn * r.c[a]});
        SegDesc sg{};
        if (kindR == K_I) {            // one-sided left: psi'[l'][r] += f O_L[l'][l] psi[l][r]
          if (r.n != 1) throw std::logic_error("one-sided run with n > 1");
          sg.a = la; sg.K = (int32_t)dL; sg.a_kn1 = FLAT; sg.a_khi = 0;
          if (!g.dagL) { sg.a_ms = (int32_t)dL; sg.a_klo = 1; } else { sg.a_ms = 1; sg.a_klo = (int32_t)dLp; }
          sg.b = mkref(B_PSI_IN, b.off); sg.b_ks = (int32_t)dR; sg.b_nlo = 1; sg.b_nhi = 0;
          sg.alpha = sgn * r.c[0];
          segs2[po->second].push_back(sg);
          segn2[po->second].push_back(1);
          P.falg += 2 * dLp * dL * dR;
          P.tab_falg_blocks[po->second] += 2 * dLp * dL * dR;
          continue;
        }
        if (kindL == K_I) {            // one-sided right: psi'[l][r'] += f psi[l][r] O_R[r'][r]
          if (r.n != 1) throw std::logic_error("one-sided run with n > 1");
          sg.a = mkref(B_PSI_IN, b.off); sg.a_ms = (int32_t)dR; sg.a_kn1 = FLAT; sg.a_klo = 1; sg.a_khi = 0;
          sg.K = (int32_t)dR;
          sg.b = ra; sg.b_nhi = 0;
          if (!g.dagR) { sg.b_ks = 1; sg.b_nlo = (int32_t)dR; } else { sg.b_ks = (int32_t)dRp; sg.b_nlo = 1; }
          sg.alpha = sgn * r.c[0];
          segs2[po->second].push_back(sg);
          segn2[po->second].push_back(1);
          P.falg += 2 * dL * dR * dRp;
          P.tab_falg_blocks[po->second] += 2 * dL * dR * dRp;
          continue;
        }
        // stage 1: T[alpha][l][r'] = f_alpha sum_r psi[l][r] O_R,alpha[r'][r]
        int64_t toff = scratch;
        scratch += (int64_t)r.n * dL * dRp;
        SegDesc s1{};
        s1.a = mkref(B_PSI_IN, b.off); s1.a_ms = (int32_t)dR; s1.a_kn1 = FLAT; s1.a_klo = 1; s1.a_khi = 0;
        s1.K = (int32_t)dR; s1.alpha = 1.0; s1.b = ra;
        if (!g.dagR) { s1.b_ks = 1; s1.b_nlo = (int32_t)dR; s1.b_nhi = dRp * dR; }
        else { s1.b_ks = (int32_t)dRp; s1.b_nlo = 1; s1.b_nhi = dR * dRp; }
        JobDesc j1{};
        j1.c = mkref(B_SCRATCH, toff); j1.scale = mkref(B_COEF, r.coef_off + (sgn < 0 ? r.n : 0));
        j1.M = (int32_t)dL; j1.N = (int32_t)(r.n * dRp); j1.c_ms = (int32_t)dRp; j1.n1 = (int32_t)dRp;
        j1.c_nlo = 1; j1.c_nhi = dL * dRp;
        j1.seg_begin = (int32_t)P.stage1.segs.size(); j1.seg_end = j1.seg_begin + 1;
        P.stage1.segs.push_back(s1);
        P.stage1.jobs.push_back(j1);
        P.falg += 2 * dL * dR * r.n * dRp;
        P.tab_falg_blocks[po->second] += 2 * dL * dR * r.n * dRp + 2 * dLp * r.n * dL * dRp;
        // stage 2: psi'[l'][r'] += sum_{alpha,l} O_L,alpha[l'][l] T[alpha][l][r']
        sg.a = la; sg.K = (int32_t)(r.n * dL); sg.alpha = 1.0;
        if (!g.dagL) { sg.a_ms = (int32_t)dL; sg.a_kn1 = (int32_t)dL; sg.a_klo = 1; sg.a_khi = dLp * dL; }
        else { sg.a_ms = 1; sg.a_kn1 = FLAT; sg.a_klo = (int32_t)dLp; sg.a_khi = 0; }
        sg.b = mkref(B_SCRATCH, toff); sg.b_ks = (int32_t)dRp; sg.b_nlo = 1; sg.b_nhi = 0;
        segs2[po->second].push_back(sg);
        segn2[po->second].push_back(r.n);
        P.falg += 2 * dLp * r.n * dL * dRp;
      }
    }
  }
  P.scratch_elems = scratch;
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
  for (size_t bi = 0; bi < P.psi.size(); ++bi) {
    const PsiBlock &b = P.psi[bi];
    // cut the segment list into pieces of at most `target` K-blocks
    std::vector<SegDesc> pieces;
    for (size_t si = 0; si < segs2[bi].size(); ++si) {
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
      }
    }
    std::vector<std::pair<int, int>> chunks;   // [begin, end) over pieces
    int64_t acc_it = 0; int begin = 0;
    for (int pi = 0; pi < (int)pieces.size(); ++pi) {
      int64_t it = (pieces[pi].K + 15) / 16;
      if (pi > begin && acc_it + it > target) { chunks.push_back({begin, pi}); begin = pi; acc_it = 0; }
      acc_it += it;
    }
    chunks.push_back({begin, (int)pieces.size()});
    const int64_t mn = b.dL * b.dR;
    const bool direct = chunks.size() == 1;
    if (!direct) {
      P.reduce.push_back(ReduceJob{b.off, P.partial_elems, (int32_t)mn, (int32_t)chunks.size()});
    }
    for (size_t c = 0; c < chunks.size(); ++c) {
      JobDesc jd{};
      jd.c = direct ? mkref(B_PSI_OUT, b.off) : mkref(B_PARTIAL, P.partial_elems + (int64_t)c * mn);
      jd.scale = -1;
      jd.M = (int32_t)b.dL; jd.N = (int32_t)b.dR; jd.c_ms = (int32_t)b.dR; jd.n1 = FLAT; jd.c_nlo = 1; jd.c_nhi = 0;
      jd.seg_begin = (int32_t)P.stage2.segs.size();
      P.stage2.segs.insert(P.stage2.segs.end(), pieces.begin() + chunks[c].first, pieces.begin() + chunks[c].second);
      jd.seg_end = (int32_t)P.stage2.segs.size();
      P.stage2.jobs.push_back(jd);
    }
    if (!direct) P.partial_elems += (int64_t)chunks.size() * mn;
    DiagJob dj{b.off, (int32_t)b.dL, (int32_t)b.dR, (int32_t)P.diag_terms.size(), 0};
    P.diag_terms.insert(P.diag_terms.end(), diag[bi].begin(), diag[bi].end());
    dj.t_end = (int32_t)P.diag_terms.size();
    P.diag_jobs.push_back(dj);
  }
  make_tiles(P.stage1, BM, BN, STRIP);
  make_tiles(P.stage2, BM, BN, 1);
  for (const Group &g : P.groups) {
    int64_t n = 0;
    for (auto &r : g.runs) n += r.n;
    int64_t row[9] = {g.s1p, g.s1, g.s2p, g.s2, Lb.classes[g.clsL].kind, g.dagL, Rb.classes[g.clsR].kind,
                      g.dagR, n};
    P.tab_groups.insert(P.tab_groups.end(), row, row + 9);
  }
  P.tab_opL = op_block_table(Lb);
  P.tab_opR = op_block_table(Rb);
  P.tab_counts = {(int64_t)P.stage1.jobs.size(), (int64_t)P.stage1.segs.size(), (int64_t)P.stage2.jobs.size(),
                  (int64_t)P.stage2.segs.size(), (int64_t)P.stage1.tiles.size(), (int64_t)P.stage2.tiles.size(),
                  P.scratch_elems, Lb.elems, Rb.elems, P.derL_elems, P.derR_elems};
}

// ----------------------------------------------------------------------------- renormalization plan
void build_renorm_plan(RenormPlan &P, const Integrals &ints, const BlockState &blk, int site,
                       bool site_is_right, const BondTable &new_tab, int L, int BM, int BN) {
  P = RenormPlan();
  P.res.ints = &ints; P.res.blk = &blk;
  BlockState &nx = P.next;
  nx.orbs = blk.orbs;
  nx.orbs.push_back(2 * site); nx.orbs.push_back(2 * site + 1);
  std::sort(nx.orbs.begin(), nx.orbs.end());
  nx.n_orb = blk.n_orb + 1;
  nx.tab = new_tab;
  layout_block(nx, L);
  P.iso = iso_blocks(blk.tab, new_tab, &P.iso_elems);
  std::map<std::pair<int, int>, std::vector<const IsoBlock *>> iso_of;   // (ip, s) -> blocks
  for (const IsoBlock &ib : P.iso) iso_of[{ib.ip, ib.s}].push_back(&ib);

  std::vector<RPiece> pieces = renorm_pieces(ints, blk.orbs, site, site_is_right, block_targets(nx));
  // group by (target class, site unit, source class, source dagger); per target member a lincomb
  struct RKey { int tcls, unit, scls, sdag; bool operator<(const RKey &o) const {
    return std::tie(tcls, unit, scls, sdag) < std::tie(o.tcls, o.unit, o.scls, o.sdag); } };
  std::map<RKey, std::map<int, std::vector<std::pair<Sym, double>>>> groups;
  for (const RPiece &p : pieces) {
    Sym ts{p.target.kind, 0, p.target.i, p.target.k};
    int tcls = nx.find_class(p.target.kind, sym_dq(ts));
    int tidx = nx.classes[tcls].member_index.at({p.target.i, p.target.k});
    int scls, sdag;
    if (!P.res.flat(p.src, &scls, &sdag, nullptr, nullptr)) continue;
    groups[RKey{tcls, p.sp * 4 + p.s, scls, sdag}][tidx].push_back({p.src, p.c});
  }
  struct RRun { int tcls, unit, scls, sdag, t0, n; OpRef src; std::vector<double> c; int64_t coef_off; };
  std::vector<RRun> runs;
  for (auto &ge : groups) {
    const RKey &k = ge.first;
    struct Al { int t; OpRef src; double c; };
    std::vector<Al> al;
    for (auto &te : ge.second) {
      int dagtmp;
      if (te.second.size() == 1) {
        al.push_back({te.first, P.res.resolve(te.second[0].first, &dagtmp), te.second[0].second});
      } else {
        std::vector<double> w(blk.classes[k.scls].n(), 0.0), wa;
        for (auto &a : te.second) {
          int c_, d_;
          P.res.flat(a.first, &c_, &d_, &wa, nullptr);
          for (size_t i = 0; i < w.size(); ++i) w[i] += a.second * wa[i];
        }
        al.push_back({te.first, P.res.resolve_weights(k.scls, w), 1.0});
      }
    }
    for (size_t a = 0; a < al.size(); ++a) {
      if (a > 0 && al[a].t == al[a - 1].t + 1 && consecutive(al[a - 1].src, al[a].src) &&
          runs.back().tcls == k.tcls && runs.back().unit == k.unit && runs.back().scls == k.scls &&
          runs.back().sdag == k.sdag && runs.back().t0 + runs.back().n == al[a].t) {
        runs.back().n++;
        runs.back().c.push_back(al[a].c);
      } else {
        runs.push_back(RRun{k.tcls, k.unit, k.scls, k.sdag, al[a].t, 1, al[a].src, {al[a].c}, 0});
      }
    }
  }
  // split runs so that target member ranges within a class are identical or disjoint
  {
    std::map<int, std::set<int>> cuts;
    for (auto &r : runs) { cuts[r.tcls].insert(r.t0); cuts[r.tcls].insert(r.t0 + r.n); }
    std::vector<RRun> split;
    for (auto &r : runs) {
      const std::set<int> &cs = cuts[r.tcls];
      int t = r.t0;
      while (t < r.t0 + r.n) {
        int nxt = *cs.upper_bound(t);
        RRun q = r;
        q.t0 = t; q.n = nxt - t;
        q.src.idx = r.src.idx + (t - r.t0);
        q.c.assign(r.c.begin() + (t - r.t0), r.c.begin() + (nxt - r.t0));
        split.push_back(q);
        t = nxt;
      }
    }
    runs.swap(split);
  }
  int64_t coefW = 0;
  P.der_elems = P.res.finalize(&coefW);
  P.res.coef_data(P.coef);
  for (auto &r : runs) {
    r.coef_off = (int64_t)P.coef.size();
    for (double c : r.c) P.coef.push_back(c);
    for (double c : r.c) P.coef.push_back(-c);
  }
  P.res.contraction_jobs(P.contract, site_is_right ? B_OPS_L : B_OPS_R, B_DER_TMP, 0);
  make_tiles(P.contract, BM, BN, STRIP);

  // --- rotation descriptors: Y = f O X_ket (rot1), O' = X_bra^T Y (rot2)
  const int buf_ops = site_is_right ? B_OPS_L : B_OPS_R;
  std::map<std::tuple<int, int, int, int>, std::vector<SegDesc>> segs2;   // (tcls, tblock, t0, n)
  int64_t scratch = 0;
  for (const RRun &r : runs) {
    const OpClass &sc = blk.classes[r.scls];
    const OpClass &tc = nx.classes[r.tcls];
    DQ dq = sc.dq;
    if (r.sdag) dq = DQ{-dq.dN, -dq.dS};
    int sp = r.unit / 4, s = r.unit % 4;
    int pis = (SITE_N[sp] - SITE_N[s]) & 1, pib = dq.dN & 1;
    for (int ik = 0; ik < (int)blk.tab.sec.size(); ++ik) {      // ket sector of the block
      const Sector &qk = blk.tab.sec[ik];
      int ib = blk.tab.find(qk.N + dq.dN, qk.S + dq.dS);       // bra sector of the block
      if (ib < 0) continue;
      auto kit = iso_of.find({ik, s});
      auto bit = iso_of.find({ib, sp});
      if (kit == iso_of.end() || bit == iso_of.end()) continue;
      int sbra = r.sdag ? ik : ib, sket = r.sdag ? ib : ik;     // stored orientation
      ref_t oa;
      if (!op_addr(P.res, r.src, buf_ops, B_DER_TMP, sbra, sket, &oa, nullptr)) continue;
      // Appendix A1: block left of site: (-1)^{N_block(ket) pi_site}; site left: (-1)^{N_site(ket) pi_block}
      int e = site_is_right ? (qk.N * pis) : (SITE_N[s] * pib);
      double sgn = (e & 1) ? -1.0 : 1.0;
      int64_t dl = qk.dim, dlp = blk.tab.sec[ib].dim;
      for (const IsoBlock *xk : kit->second)
        for (const IsoBlock *xb : bit->second) {
          auto tb = tc.block_index.find({xb->in, xk->in});
          if (tb == tc.block_index.end()) continue;
          int64_t dA = xk->cols, dAp = xb->cols;
          int64_t yoff = scratch;
          scratch += (int64_t)r.n * dlp * dA;
          // rot1: Y[alpha][l'][a] = f_alpha sum_l O_alpha[l'][l] X_k[l][a];  m = a, n = (alpha, l')
          SegDesc s1{};
          s1.a = mkref(B_ISO, xk->off); s1.a_ms = 1; s1.a_kn1 = FLAT; s1.a_klo = (int32_t)dA; s1.a_khi = 0;
          s1.K = (int32_t)dl; s1.alpha = 1.0; s1.b = oa;
          if (!r.sdag) { s1.b_ks = 1; s1.b_nlo = (int32_t)dl; s1.b_nhi = dlp * dl; }
          else { s1.b_ks = (int32_t)dlp; s1.b_nlo = 1; s1.b_nhi = dl * dlp; }
          JobDesc j1{};
          j1.c = mkref(B_SCRATCH, yoff); j1.scale = mkref(B_COEF, r.coef_off + (sgn < 0 ? r.n : 0));
          j1.M = (int32_t)dA; j1.N = (int32_t)(r.n * dlp); j1.c_ms = 1; j1.n1 = (int32_t)dlp;
          j1.c_nlo = (int32_t)dA; j1.c_nhi = dlp * dA;
          j1.seg_begin = (int32_t)P.rot1.segs.size(); j1.seg_end = j1.seg_begin + 1;
          P.rot1.segs.push_back(s1);
          P.rot1.jobs.push_back(j1);
          P.rot1.flops += 2 * dA * dl * r.n * dlp;
          // rot2: O'[alpha][a'][a] += sum_l' X_b[l'][a'] Y[alpha][l'][a];  m = a', n = (alpha, a)
          SegDesc s2{};
          s2.a = mkref(B_ISO, xb->off); s2.a_ms = 1; s2.a_kn1 = FLAT; s2.a_klo = (int32_t)dAp; s2.a_khi = 0;
          s2.K = (int32_t)dlp; s2.alpha = 1.0;
          s2.b = mkref(B_SCRATCH, yoff); s2.b_ks = (int32_t)dA; s2.b_nlo = 1; s2.b_nhi = dlp * dA;
          segs2[std::make_tuple(r.tcls, tb->second, r.t0, r.n)].push_back(s2);
          P.rot2.flops += 2 * dAp * dlp * r.n * dA;
        }
    }
  }
  P.scratch_elems = scratch;
  for (auto &e : segs2) {
    int tcls, tblk, t0, n;
    std::tie(tcls, tblk, t0, n) = e.first;
    const OpClass &tc = nx.classes[tcls];
    const OpBlock &ob = tc.blocks[tblk];
    int64_t dAp = nx.tab.sec[ob.bra].dim, dA = nx.tab.sec[ob.ket].dim;
    JobDesc jd{};
    jd.c = mkref(B_NEW, ob.off + (int64_t)t0 * dAp * dA); jd.scale = -1;
    jd.M = (int32_t)dAp; jd.N = (int32_t)(n * dA); jd.c_ms = (int32_t)dA; jd.n1 = (int32_t)dA;
    jd.c_nlo = 1; jd.c_nhi = dAp * dA;
    jd.seg_begin = (int32_t)P.rot2.segs.size();
    P.rot2.segs.insert(P.rot2.segs.end(), e.second.begin(), e.second.end());
    jd.seg_end = (int32_t)P.rot2.segs.size();
    P.rot2.jobs.push_back(jd);
  }
  make_tiles(P.rot1, BM, BN, STRIP);
  make_tiles(P.rot2, BM, BN, 1);
}

}  // namespace dmrg
