// Renormalization plan (Appendix A3/A4/A5): every operator of the grown block
// is a sum of pieces  f X_bra^T (O_src (x) site unit) X_ket;  rot1 forms Y = c O_src X_ket per source
// block and ket pair, rot2 accumulates G X_bra^T Y into the new block (output-stationary).
// G: fermion sign (U(1)xU(1)) or 9j prefactor, sign and tilde factor (SU(2)).
#include <algorithm>
#include <cmath>
#include <stdexcept>

#include "internal.h"

namespace dmrg {

namespace {
inline double tilde_factor(int S_bra, int S_ket, int k2) {   // <bra||T~||ket> = factor * <ket||T||bra>
  int e = (S_ket - S_bra + k2) / 2;
  return ((e & 1) ? -1.0 : 1.0) * std::sqrt((S_ket + 1.0) / (S_bra + 1.0));
}
}  // namespace

void build_renorm_plan(RenormPlan &P, const Integrals &ints, const BlockState &blk, int site,
                       bool site_is_right, const BondTable &new_tab, int L, int BM, int BN, bool emu,
                       const PlanOptions *opt) {
  P = RenormPlan();
  if (emu) {
    P.emu = std::make_shared<HeffPlan>();
    P.emu->emu_mode = true;
    if (opt) P.emu->opt = *opt;
    P.emu->emu.assign(1, EmuPass());
  }
  HeffPlan *E = P.emu.get();
  auto pad = [](int64_t x, int64_t r) { return (x + r - 1) / r * r; };
  std::map<std::tuple<ref_t, int, int>, std::pair<int64_t, int64_t>> op_units;   // operator unit -> (out_off, exp_off) in sliceR
  std::map<int64_t, std::pair<int64_t, int64_t>> xk_units, xb_units;             // isometry block offset -> unit (sliceP / sliceT)
  std::map<std::tuple<int, int, int, int>, std::vector<EmuSeg>> esegs2;
  // a 64-row unit of isometry columns: X[l][a] row-major, line a, K = l
  auto x_unit = [&](const IsoBlock *x, std::vector<EmuSliceDesc> &list, int64_t &bytes, int64_t &nexp,
                    std::map<int64_t, std::pair<int64_t, int64_t>> &seen) {
    auto it = seen.find(x->off);
    if (it != seen.end()) return it->second;
    EmuSliceDesc d{};
    d.src = mkref(B_ISO, x->off); d.lstride = x->cols; d.linestride = 1; d.n_members = 1;
    d.dl = d.dlpad = (int32_t)x->rows; d.lines = (int32_t)x->cols; d.ld = pad(x->rows, 32); d.tile_rows = 64;
    d.out_off = bytes; d.exp_off = nexp;
    bytes += pad(x->cols, 64) * d.ld; nexp += pad(x->cols, 4);
    list.push_back(d);
    return seen.emplace(x->off, std::make_pair(d.out_off, d.exp_off)).first->second;
  };
  const int sym = blk.sym;
  P.res.ints = &ints; P.res.blk = &blk;
  BlockState &nx = P.next;
  nx.sym = sym;
  nx.orbs = blk.orbs;
  if (sym == 0) { nx.orbs.push_back(2 * site); nx.orbs.push_back(2 * site + 1); } else nx.orbs.push_back(site);
  std::sort(nx.orbs.begin(), nx.orbs.end());
  nx.n_orb = blk.n_orb + 1;
  nx.tab = new_tab;
  layout_block(nx, L);
  P.iso = iso_blocks(blk.tab, new_tab, sym, &P.iso_elems);
  std::map<std::pair<int, int>, std::vector<const IsoBlock *>> iso_of;   // (ip, s) -> blocks
  for (const IsoBlock &ib : P.iso) iso_of[{ib.ip, ib.s}].push_back(&ib);

  // targets with their ranks
  std::vector<OpKey> targets;
  for (const OpClass &c : nx.classes)
    for (auto &m : c.members) {
      OpKey k{c.kind, m.first, m.second, 0};
      if (sym != 0 && (c.kind == K_A || c.kind == K_B)) k.rank = c.dq.dS;
      targets.push_back(k);
    }
  std::vector<RPiece> pieces = sym == 0 ? renorm_pieces(ints, blk.orbs, site, site_is_right, targets)
                                        : renorm_pieces_su2(ints, blk.orbs, site, site_is_right, targets);
  struct RKey { int tcls, unit, scls, sdag, kS; bool operator<(const RKey &o) const {
    return std::tie(tcls, unit, scls, sdag, kS) < std::tie(o.tcls, o.unit, o.scls, o.sdag, o.kS); } };
  std::map<RKey, std::map<int, std::map<Sym, double>>> groups;   // per target member: lincomb of source symbols
  for (const RPiece &p : pieces) {
    Sym ts{p.target.kind, 0, p.target.i, p.target.k};
    ts.rank = p.target.rank;
    int tcls = nx.find_class(p.target.kind, sym_class(ts, sym));
    if (tcls < 0) throw std::logic_error("renormalization target without a class");
    int tidx = nx.classes[tcls].member_index.at({p.target.i, p.target.k});
    int scls, sdag;
    if (!P.res.flat(p.src, &scls, &sdag, nullptr, nullptr)) continue;
    groups[RKey{tcls, p.sp * 4 + p.s, scls, sdag, p.kS}][tidx][p.src] += p.c;
  }
  struct RRun { int tcls, unit, scls, sdag, kS, t0, n; OpRef src; std::vector<double> c; int64_t coef_off; };
  std::vector<RRun> runs;
  for (auto &ge : groups) {
    const RKey &k = ge.first;
    struct Al { int t; OpRef src; double c; };
    std::vector<Al> al;
    for (auto &te : ge.second) {
      int dagtmp;
      std::vector<std::pair<Sym, double>> lc;
      for (auto &x : te.second) if (x.second != 0.0) lc.push_back(x);
      if (lc.empty()) continue;
      if (lc.size() == 1) {
        al.push_back({te.first, P.res.resolve(lc[0].first, &dagtmp), lc[0].second});
      } else {
        std::vector<double> w(blk.classes[k.scls].n(), 0.0), wa;
        for (auto &a : lc) {
          int c_, d_;
          P.res.flat(a.first, &c_, &d_, &wa, nullptr);
          for (size_t i = 0; i < w.size(); ++i) w[i] += a.second * wa[i];
        }
        al.push_back({te.first, P.res.resolve_weights(k.scls, w), 1.0});
      }
    }
    bool fresh = true;
    for (size_t a = 0; a < al.size(); ++a) {
      if (!fresh && al[a].t == al[a - 1].t + 1 && consecutive(al[a - 1].src, al[a].src)) {
        runs.back().n++;
        runs.back().c.push_back(al[a].c);
      } else {
        runs.push_back(RRun{k.tcls, k.unit, k.scls, k.sdag, k.kS, al[a].t, 1, al[a].src, {al[a].c}, 0});
        fresh = false;
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
  }
  const int buf_ops = site_is_right ? B_OPS_L : B_OPS_R;
  P.res.contraction_jobs(P.contract, buf_ops, B_DER_TMP, 0);
  make_tiles(P.contract, BM, BN, STRIP);

  std::map<std::tuple<int, int, int, int>, std::vector<SegDesc>> segs2;   // (tcls, tblock, t0, n)
  std::map<int64_t, std::pair<int64_t, int64_t>> y_units;                 // yoff -> unit in sliceL
  int64_t scratch = 0;
  for (const RRun &r : runs) {
    const OpClass &sc = blk.classes[r.scls];
    const OpClass &tc = nx.classes[r.tcls];
    const int kB = sc.dq.dS, K = tc.dq.dS;             // SU(2): doubled ranks of source and target
    const int sp = r.unit / 4, s = r.unit % 4;
    const int pis = (site_N(sym, sp) - site_N(sym, s)) & 1, pib = sc.dq.dN & 1;
    for (int ik = 0; ik < (int)blk.tab.sec.size(); ++ik) {      // ket sector of the block
      const Sector &qk = blk.tab.sec[ik];
      auto kit = iso_of.find({ik, s});
      if (kit == iso_of.end()) continue;
      // bra sectors of the block reachable through the (possibly daggered) source class
      std::vector<int> bras;
      const int dN = r.sdag ? -sc.dq.dN : sc.dq.dN;
      if (sym == 0) {
        int i = blk.tab.find(qk.N + dN, qk.S + (r.sdag ? -sc.dq.dS : sc.dq.dS));
        if (i >= 0) bras.push_back(i);
      } else {
        for (int S2 = std::abs(qk.S - kB); S2 <= qk.S + kB; S2 += 2) {
          int i = blk.tab.find(qk.N + dN, S2);
          if (i >= 0) bras.push_back(i);
        }
      }
      for (int ib : bras) {
        auto bit = iso_of.find({ib, sp});
        if (bit == iso_of.end()) continue;
        const Sector &qb = blk.tab.sec[ib];
        int sbra = r.sdag ? ik : ib, sket = r.sdag ? ib : ik;     // stored orientation
        ref_t oa;
        if (!op_addr(P.res, r.src, buf_ops, B_DER_TMP, sbra, sket, &oa, nullptr)) continue;
        const int64_t dl = qk.dim, dlp = qb.dim;
        for (const IsoBlock *xk : kit->second) {
          int64_t yoff = -1;
          const int64_t dA = xk->cols;
          for (const IsoBlock *xb : bit->second) {
            auto tb = tc.block_index.find({xb->in, xk->in});
            if (tb == tc.block_index.end()) continue;
            double G;
            if (sym == 0) {   // Appendix A1: block left of site (-1)^{N_block pi_site}; site left (-1)^{N_site pi_block}
              int e = site_is_right ? (qk.N * pis) : (site_N(sym, s) * pib);
              G = (e & 1) ? -1.0 : 1.0;
            } else {
              const int SA = new_tab.sec[xk->in].S, SAp = new_tab.sec[xb->in].S;
              G = site_is_right
                      ? su2_f9(qk.S, site_S(sym, s), SA, kB, r.kS, K, qb.S, site_S(sym, sp), SAp)
                      : su2_f9(site_S(sym, s), qk.S, SA, r.kS, kB, K, site_S(sym, sp), qb.S, SAp);
              if (G == 0.0) continue;
              int e = site_is_right ? (qk.N * pis) : (site_N(sym, s) * pib);
              if (e & 1) G = -G;
              if (r.sdag) G *= tilde_factor(qb.S, qk.S, kB);
            }
            const int64_t dAp = xb->cols;
            if (yoff < 0) {   // rot1: Y[alpha][l'][a] = c_alpha sum_l O_alpha[l'][l] X_k[l][a];  m = a, n = (alpha, l')
              yoff = scratch;
              scratch += (int64_t)r.n * dlp * dA;
              SegDesc s1{};
              s1.a = mkref(B_ISO, xk->off); s1.a_ms = 1; s1.a_kn1 = FLAT; s1.a_klo = (int32_t)dA; s1.a_khi = 0;
              s1.K = (int32_t)dl; s1.alpha = 1.0; s1.b = oa;
              if (!r.sdag) { s1.b_ks = 1; s1.b_nlo = (int32_t)dl; s1.b_nhi = dlp * dl; }
              else { s1.b_ks = (int32_t)dlp; s1.b_nlo = 1; s1.b_nhi = dl * dlp; }
              JobDesc j1{};
              j1.c = mkref(B_SCRATCH, yoff); j1.scale = mkref(B_COEF, r.coef_off);
              j1.M = (int32_t)dA; j1.N = (int32_t)(r.n * dlp); j1.c_ms = 1; j1.n1 = (int32_t)dlp;
              j1.c_nlo = (int32_t)dA; j1.c_nhi = dlp * dA;
              j1.seg_begin = (int32_t)P.rot1.segs.size(); j1.seg_end = j1.seg_begin + 1;
              P.rot1.segs.push_back(s1);
              P.rot1.jobs.push_back(j1);
              P.rot1.flops += 2 * dA * dl * r.n * dlp;
              if (E) {   // rot1 on the tensor cores: rows = operator lines (alpha, l'), columns = a, K = l; Y[alpha][a][l']
                const int64_t kpad = pad(dl, 32), nlines = (int64_t)r.n * dlp;
                auto key = std::make_tuple(oa, (int)r.sdag, r.n);
                auto ou = op_units.find(key);
                if (ou == op_units.end()) {
                  ou = op_units.emplace(key, std::make_pair(E->emuR_bytes, E->expR_n)).first;
                  EmuSliceDesc d{};
                  d.n_members = 1; d.dl = d.dlpad = (int32_t)dl; d.ld = kpad; d.tile_rows = 128;
                  d.out_off = E->emuR_bytes; d.exp_off = E->expR_n;
                  if (!r.sdag) {              // stored [member][l'][l]: the lines are contiguous rows
                    d.src = oa; d.lstride = 1; d.linestride = dl; d.lines = (int32_t)nlines;
                    E->sliceR.push_back(d);
                  } else {                    // stored [member][l][l']: one descriptor per member
                    d.lstride = dlp; d.linestride = 1; d.lines = (int32_t)dlp;
                    for (int a = 0; a < r.n; ++a) {
                      d.src = oa + (int64_t)a * dl * dlp; d.line_base = (int32_t)(a * dlp);
                      E->sliceR.push_back(d);
                    }
                  }
                  E->emuR_bytes += pad(nlines, 128) * kpad; E->expR_n += nlines;
                }
                auto xu = x_unit(xk, E->sliceP, E->emuP_bytes, E->expP_n, xk_units);
                EmuPass &EP = E->emu[0];
                EmuSeg es{};
                es.a_off = ou->second.first; es.ea_off = ou->second.second; es.b_off = xu.first; es.eb_off = xu.second;
                es.ksteps = (int32_t)(kpad / 32); es.alpha = 1.0;
                EmuJob ej{};
                ej.c = mkref(B_SCRATCH, yoff); ej.scale = mkref(B_COEF, r.coef_off); ej.c_nhi = dA * dlp;
                ej.M = (int32_t)nlines; ej.N = (int32_t)dA; ej.c_ld = (int32_t)dlp; ej.n1 = (int32_t)dlp; ej.rows_split = 1;
                ej.seg_begin = (int32_t)EP.segs1.size(); ej.seg_end = ej.seg_begin + 1;
                EP.segs1.push_back(es);
                for (int m0 = 0; m0 < ej.M; m0 += 128)
                  for (int n0 = 0; n0 < ej.N; n0 += 64) EP.tiles1.push_back(EmuTile{(int32_t)EP.jobs1.size(), m0, n0, 1});
                EP.jobs1.push_back(ej);
                E->flops_emu1 += 2 * dA * dl * r.n * dlp;
              }
            }
            // rot2: O'[alpha][a'][a] += G sum_l' X_b[l'][a'] Y[alpha][l'][a];  m = a', n = (alpha, a)
            SegDesc s2{};
            s2.a = mkref(B_ISO, xb->off); s2.a_ms = 1; s2.a_kn1 = FLAT; s2.a_klo = (int32_t)dAp; s2.a_khi = 0;
            s2.K = (int32_t)dlp; s2.alpha = G;
            s2.b = mkref(B_SCRATCH, yoff); s2.b_ks = (int32_t)dA; s2.b_nlo = 1; s2.b_nhi = dlp * dA;
            segs2[std::make_tuple(r.tcls, tb->second, r.t0, r.n)].push_back(s2);
            P.rot2.flops += 2 * dAp * dlp * r.n * dA;
            if (E) {     // rot2: rows = lines (alpha, a) of Y, K = l' contiguous; columns = a' of X_b
              auto yu = y_units.find(yoff);
              if (yu == y_units.end()) {
                EmuSliceDesc d{};
                d.src = mkref(B_SCRATCH, yoff); d.lstride = 1; d.linestride = dlp; d.n_members = 1;
                d.dl = d.dlpad = (int32_t)dlp; d.lines = (int32_t)(r.n * dA); d.ld = pad(dlp, 32); d.tile_rows = 128;
                d.out_off = E->emuL_bytes; d.exp_off = E->expL_n;
                E->emuL_bytes += pad((int64_t)r.n * dA, 128) * d.ld; E->expL_n += (int64_t)r.n * dA;
                E->sliceL.push_back(d);
                yu = y_units.emplace(yoff, std::make_pair(d.out_off, d.exp_off)).first;
              }
              auto xu = x_unit(xb, E->emu[0].sliceT, E->emuT_bytes, E->expT_n, xb_units);
              EmuSeg es{};
              es.a_off = yu->second.first; es.ea_off = yu->second.second; es.b_off = xu.first; es.eb_off = xu.second;
              es.ksteps = (int32_t)(pad(dlp, 32) / 32); es.alpha = G;
              esegs2[std::make_tuple(r.tcls, tb->second, r.t0, r.n)].push_back(es);
              E->flops_emu += 2 * dAp * dlp * r.n * dA;
            }
          }
        }
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
    if (E) {
      EmuPass &EP = E->emu[0];
      EmuJob ej{};
      ej.c = jd.c; ej.scale = -1; ej.c_nhi = dAp * dA; ej.M = (int32_t)(n * dA); ej.N = (int32_t)dAp;
      ej.c_ld = (int32_t)dA; ej.n1 = (int32_t)dA; ej.rows_split = 1;
      ej.seg_begin = (int32_t)EP.segs.size();
      const auto &v = esegs2[e.first];
      EP.segs.insert(EP.segs.end(), v.begin(), v.end());
      ej.seg_end = (int32_t)EP.segs.size();
      for (int m0 = 0; m0 < ej.M; m0 += 128)
        for (int n0 = 0; n0 < ej.N; n0 += 64) EP.tiles.push_back(EmuTile{(int32_t)EP.jobs.size(), m0, n0, 1});
      EP.jobs.push_back(ej);
    }
  }
  make_tiles(P.rot1, BM, BN, STRIP);
  make_tiles(P.rot2, BM, BN, 1);
}

}  // namespace dmrg
