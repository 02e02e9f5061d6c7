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

int n_site_states(int sym) { return sym == 0 ? 4 : 3; }
int site_N(int sym, int s) { static const int n3[3] = {0, 1, 2}; return sym == 0 ? SITE_N[s] : n3[s]; }
int site_S(int sym, int s) { static const int j3[3] = {0, 1, 0}; return sym == 0 ? SITE_S[s] : j3[s]; }
// second labels reachable by fusing a block label S with site state s (one value for U(1)xU(1))
std::vector<int> fuse_S(int sym, int S, int s) {
  if (sym == 0) return {S + SITE_S[s]};
  std::vector<int> r;
  int j = site_S(sym, s);
  for (int x = std::abs(S - j); x <= S + j; x += 2) r.push_back(x);
  return r;
}

std::vector<IsoBlock> iso_blocks(const BondTable &prev, const BondTable &next, int sym, int64_t *total) {
  std::vector<IsoBlock> out;
  int64_t off = 0;
  for (int ip = 0; ip < (int)prev.sec.size(); ++ip)
    for (int s = 0; s < n_site_states(sym); ++s) {
      std::vector<int> ins;
      for (int S2 : fuse_S(sym, prev.sec[ip].S, s)) {
        int in = next.find(prev.sec[ip].N + site_N(sym, s), S2);
        if (in >= 0) ins.push_back(in);
      }
      std::sort(ins.begin(), ins.end());
      for (int in : ins) {
        IsoBlock b{ip, s, in, prev.sec[ip].dim, next.sec[in].dim, off};
        off += b.rows * b.cols;
        out.push_back(b);
      }
    }
  if (total) *total = off;
  return out;
}

// ----------------------------------------------------------------------------- layouts
void layout_block(BlockState &b, int L) {
  b.classes.clear();
  b.class_index.clear();
  std::vector<char> in(2 * L + 2, 0);
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
  auto add = [&](int kind, int i, int k, int rank = 0) {
    Sym s{kind, 0, i, k};
    s.rank = rank;
    OpClass &c = cls(kind, sym_class(s, b.sym));
    c.member_index[{i, k}] = c.n();
    c.members.push_back({i, k});
  };
  add(K_I, -1, -1);
  const int n_index = b.sym == 0 ? 2 * L : L;      // spin-orbitals or spatial orbitals
  if (!b.orbs.empty()) {
    add(K_H, -1, -1);
    for (int i : b.orbs) add(K_C, i, -1);
    for (int x = 0; x < n_index; ++x) if (!in[x]) add(K_S, x, -1);
    if (b.sym == 0) {
      for (size_t a = 0; a < b.orbs.size(); ++a)
        for (size_t c = a + 1; c < b.orbs.size(); ++c) add(K_A, b.orbs[a], b.orbs[c]);
      for (int i : b.orbs) for (int l : b.orbs) add(K_B, i, l);
    } else {   // A^0_pr (p <= r), A^1_pr (p < r), B^k_ps (all p, s), SURVEY.md Appendix A4
      for (size_t a = 0; a < b.orbs.size(); ++a)
        for (size_t c = a; c < b.orbs.size(); ++c) {
          add(K_A, b.orbs[a], b.orbs[c], 0);
          if (c > a) add(K_A, b.orbs[a], b.orbs[c], 2);
        }
      for (int i : b.orbs) for (int l : b.orbs) { add(K_B, i, l, 0); add(K_B, i, l, 2); }
    }
  }
  int64_t off = 0;
  for (OpClass &c : b.classes) {
    for (int ket = 0; ket < (int)b.tab.sec.size(); ++ket) {
      const Sector &qk = b.tab.sec[ket];
      if (b.sym == 0) {
        int bra = b.tab.find(qk.N + c.dq.dN, qk.S + c.dq.dS);
        if (bra >= 0) c.blocks.push_back({bra, ket, 0});
      } else {   // triangle rule: |S - k| <= S' <= S + k
        for (int S2 = std::abs(qk.S - c.dq.dS); S2 <= qk.S + c.dq.dS; S2 += 2) {
          int bra = b.tab.find(qk.N + c.dq.dN, S2);
          if (bra >= 0) c.blocks.push_back({bra, ket, 0});
        }
      }
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
  if (b.sym != 0 && (s.kind == K_P || s.kind == K_Q)) {
    // P~^k_pr = sum_{q,s} (pq|rs) A~^k_qs over stored pairs q <= s;
    // Q~^0_ps = sum [2(ps|qr) - (pr|qs)] B^0_qr, Q~^1_ps = sum (pr|qs) B^1_qr
    auto vv = [&](int p, int q, int r, int t) {
      return ints->V[(((size_t)p * ints->L + q) * ints->L + r) * ints->L + t]; };
    const bool isP = s.kind == K_P;
    int c = b.find_class(isP ? K_A : K_B, DQ{isP ? 2 : 0, s.rank});
    if (c < 0) return false;
    *cls = c; *dag = isP ? !s.dag : 0;
    if (w) {
      const OpClass &oc = b.classes[c];
      w->assign(oc.n(), 0.0);
      const double sg = s.rank == 2 ? -1.0 : 1.0;
      for (int a = 0; a < oc.n(); ++a) {
        int q = oc.members[a].first, t = oc.members[a].second;
        if (isP) (*w)[a] = q == t ? vv(s.i, q, s.k, q) : vv(s.i, q, s.k, t) + sg * vv(s.i, t, s.k, q);
        else (*w)[a] = s.rank == 0 ? 2.0 * vv(s.i, s.k, q, t) - vv(s.i, t, q, s.k) : vv(s.i, t, q, s.k);
      }
    }
    return true;
  }
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
  int c = b.find_class(s.kind, sym_class(u, b.sym));
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
bool op_addr(const Resolver &res, const OpRef &r, int buf_ops, int buf_der, int bra, int ket,
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

bool consecutive(const OpRef &a, const OpRef &b) {
  return a.derived == b.derived && a.arr == b.arr && b.idx == a.idx + 1;
}

}  // namespace dmrg
