// Symbolic expansion of the ab initio Hamiltonian into (block operator) x (site operator)
// products: cut identity and blocking rules of SURVEY.md Appendix A2/A3 with the fermion
// sign rule of Appendix A1 (PAPER.md:41 fixes only the site basis; readings s1-s5).
//
// Everything here is bookkeeping over symbols and 4x4 site matrices; the numeric block
// operators never leave the device.
#include "internal.h"

#include <algorithm>
#include <cmath>
#include <stdexcept>

namespace dmrg {

const int SITE_N[4] = {0, 1, 1, 2};
const int SITE_S[4] = {0, 1, -1, 0};

// ------------------------------------------------------------------ 4x4 site algebra
static Mat4 mat_zero() { Mat4 m; m.fill(0.0); return m; }
static Mat4 mat_eye() { Mat4 m = mat_zero(); for (int s = 0; s < 4; ++s) m[s * 4 + s] = 1.0; return m; }
static Mat4 mat_mul(const Mat4 &a, const Mat4 &b) {
  Mat4 c = mat_zero();
  for (int r = 0; r < 4; ++r)
    for (int k = 0; k < 4; ++k) {
      double x = a[r * 4 + k];
      if (x == 0.0) continue;
      for (int q = 0; q < 4; ++q) c[r * 4 + q] += x * b[k * 4 + q];
    }
  return c;
}
static Mat4 mat_T(const Mat4 &a) {
  Mat4 c;
  for (int r = 0; r < 4; ++r) for (int q = 0; q < 4; ++q) c[r * 4 + q] = a[q * 4 + r];
  return c;
}
static void mat_axpy(Mat4 &y, double a, const Mat4 &x) { for (int e = 0; e < 16; ++e) y[e] += a * x[e]; }
static bool mat_is_zero(const Mat4 &a) { for (double x : a) if (x != 0.0) return false; return true; }

// a+_up, a+_dn in the basis 0=|0>, 1=|u>, 2=|d>, 3=|ud> = a+_u a+_d |0>  (Appendix A1):
// a+_u|0>=|u>, a+_u|d>=|ud>, a+_d|0>=|d>, a+_d|u> = a+_d a+_u|0> = -|ud>.
static Mat4 site_creator(int sigma) {
  Mat4 m = mat_zero();
  if (sigma == 0) { m[1 * 4 + 0] = 1.0; m[3 * 4 + 2] = 1.0; }
  else { m[2 * 4 + 0] = 1.0; m[3 * 4 + 1] = -1.0; }
  return m;
}

// ------------------------------------------------------------------ symbols
DQ sym_dq(const Sym &s) {
  DQ q{0, 0};
  switch (s.kind) {
    case K_I: case K_H: break;
    case K_C: q = {1, spin_of(s.i)}; break;
    case K_S: q = {-1, -spin_of(s.i)}; break;
    case K_A: q = {2, spin_of(s.i) + spin_of(s.k)}; break;
    case K_B: q = {0, spin_of(s.i) - spin_of(s.k)}; break;
    case K_P: q = {-2, -spin_of(s.i) - spin_of(s.k)}; break;
    case K_Q: q = {0, spin_of(s.k) - spin_of(s.i)}; break;
  }
  if (s.dag) { q.dN = -q.dN; q.dS = -q.dS; }
  return q;
}
Sym sym_dagger(const Sym &s) {
  Sym r = s;
  switch (s.kind) {
    case K_I: case K_H: break;
    case K_B: case K_Q: std::swap(r.i, r.k); break;   // (a+_i a_l)+ = a+_l a_i; (Q_il)+ = Q_li
    default: r.dag = !s.dag;
  }
  return r;
}
static LinComb lc_dagger(const LinComb &a) {
  LinComb r;
  for (auto &t : a) r.push_back({sym_dagger(t.first), t.second});
  return r;
}
static Fac fac_dagger(const Fac &f) {
  Fac r;
  r.is_site = f.is_site;
  if (f.is_site) r.m = mat_T(f.m); else r.lc = lc_dagger(f.lc);
  return r;
}
static Fac fac_sym(int kind, int i, int k, double c = 1.0) {
  Fac f; f.is_site = false; f.lc.push_back({Sym{kind, 0, i, k}, c}); return f;
}
static Fac fac_empty() { Fac f; f.is_site = false; return f; }
static Fac fac_site(const Mat4 &m) { Fac f; f.is_site = true; f.m = m; return f; }

// ------------------------------------------------------------------ parts
Part make_site_part(const Integrals *ints, int p) {
  Part P; P.is_site = true; P.p = p; P.ints = ints;
  P.orbs = {2 * p, 2 * p + 1};
  P.inside.assign(2 * ints->L, 0);
  P.inside[2 * p] = P.inside[2 * p + 1] = 1;
  return P;
}
Part make_block_part(const Integrals *ints, const std::vector<int> &orbs) {
  Part P; P.is_site = false; P.ints = ints; P.orbs = orbs;
  std::sort(P.orbs.begin(), P.orbs.end());
  P.inside.assign(2 * ints->L, 0);
  for (int i : P.orbs) P.inside[i] = 1;
  return P;
}

Fac Part::op(const OpKey &key) const {
  if (!is_site) {
    // A block answers with symbols of its stored normal set or of the complements P, Q
    // (Appendix A2).  An empty block (vacuum) has only the identity.
    bool empty = orbs.empty();
    switch (key.kind) {
      case K_I: return fac_sym(K_I, -1, -1);
      case K_H: return empty ? fac_empty() : fac_sym(K_H, -1, -1);
      case K_C: return fac_sym(K_C, key.i, -1);
      case K_S: return empty ? fac_empty() : fac_sym(K_S, key.i, -1);
      case K_A:
        if (key.i == key.k) return fac_empty();
        return key.i < key.k ? fac_sym(K_A, key.i, key.k) : fac_sym(K_A, key.k, key.i, -1.0);
      case K_B: return fac_sym(K_B, key.i, key.k);
      case K_P:  // P_ik = -P_ki; needs at least two orbitals inside
        if (key.i == key.k || orbs.size() < 2) return fac_empty();
        return key.i < key.k ? fac_sym(K_P, key.i, key.k) : fac_sym(K_P, key.k, key.i, -1.0);
      case K_Q: return empty ? fac_empty() : fac_sym(K_Q, key.i, key.k);
    }
    throw std::logic_error("bad op key");
  }
  // A site answers with the explicit 4x4 matrix of the Appendix-A2 definition.
  const Integrals &I = *ints;
  Mat4 cr[2] = {site_creator(0), site_creator(1)};
  Mat4 an[2] = {mat_T(cr[0]), mat_T(cr[1])};
  auto C = [&](int i) -> const Mat4 & { return cr[i & 1]; };
  auto Aop = [&](int i) -> const Mat4 & { return an[i & 1]; };
  Mat4 out = mat_zero();
  switch (key.kind) {
    case K_I: return fac_site(mat_eye());
    case K_C: return fac_site(C(key.i));
    case K_A: return fac_site(mat_mul(C(key.i), C(key.k)));
    case K_B: return fac_site(mat_mul(C(key.i), Aop(key.k)));
    case K_H:
      for (int i : orbs) for (int j : orbs) {
        mat_axpy(out, I.t(i, j), mat_mul(C(i), Aop(j)));
        for (int k : orbs) for (int l : orbs) {
          double w = I.v(i, j, k, l);
          if (w != 0.0) mat_axpy(out, 0.5 * w, mat_mul(mat_mul(C(i), C(k)), mat_mul(Aop(l), Aop(j))));
        }
      }
      return fac_site(out);
    case K_S: {  // S_x = 1/2 sum_j t_xj a_j + sum_jkl v_xjkl a+_k a_l a_j
      int x = key.i;
      for (int j : orbs) {
        mat_axpy(out, 0.5 * I.t(x, j), Aop(j));
        for (int k : orbs) for (int l : orbs) {
          double w = I.v(x, j, k, l);
          if (w != 0.0) mat_axpy(out, w, mat_mul(C(k), mat_mul(Aop(l), Aop(j))));
        }
      }
      return fac_site(out);
    }
    case K_P:  // P_ik = sum_jl v_ijkl a_l a_j
      for (int j : orbs) for (int l : orbs) {
        double w = I.v(key.i, j, key.k, l);
        if (w != 0.0) mat_axpy(out, w, mat_mul(Aop(l), Aop(j)));
      }
      return fac_site(out);
    case K_Q:  // Q_il = sum_kj (v_ilkj - v_ijkl) a+_k a_j
      for (int k : orbs) for (int j : orbs) {
        double w = I.v(key.i, key.k, k, j) - I.v(key.i, j, k, key.k);
        if (w != 0.0) mat_axpy(out, w, mat_mul(C(k), Aop(j)));
      }
      return fac_site(out);
  }
  throw std::logic_error("bad op key");
}

// ------------------------------------------------------------------ two-part operators
void Op2::add(const Sym &s, const Mat4 &mat, double c) {
  if (c == 0.0 || mat_is_zero(mat)) return;
  auto it = m.find(s.key());
  if (it == m.end()) {
    Mat4 z = mat_zero();
    mat_axpy(z, c, mat);
    m.emplace(s.key(), std::make_pair(s, z));
  } else {
    mat_axpy(it->second.second, c, mat);
  }
}

// out += coef * x (x) y, x on the left part; exactly one factor is the site.
static void tensor(Op2 &out, const Fac &x, const Fac &y, double coef) {
  const Fac &blk = x.is_site ? y : x;
  const Fac &site = x.is_site ? x : y;
  if (blk.is_site || !site.is_site) throw std::logic_error("tensor: need one block and one site factor");
  for (auto &t : blk.lc) out.add(t.first, site.m, coef * t.second);
}

// (X Y)+ = Y+ X+ = (-1)^{pi_X pi_Y} X+ Y+ ; the parity of the site factor is read per element.
Op2 op2_dagger(const Op2 &o) {
  Op2 r;
  for (auto &e : o.m) {
    const Sym &s = e.second.first;
    int pis = sym_dq(s).dN & 1;
    Mat4 t = mat_zero();
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
      double x = e.second.second[a * 4 + b];
      if (x == 0.0) continue;
      int pim = (SITE_N[a] - SITE_N[b]) & 1;
      t[b * 4 + a] = (pis && pim) ? -x : x;
    }
    r.add(sym_dagger(s), t, 1.0);
  }
  return r;
}

std::vector<int> Composite::orbs() const {
  std::vector<int> o = X.orbs;
  o.insert(o.end(), Y.orbs.begin(), Y.orbs.end());
  std::sort(o.begin(), o.end());
  return o;
}

struct CutTerm { double c; Fac x, y; };
// Cross terms of the cut identity (Appendix A2) for X | Y, each already in left-to-right
// order; the reorder signs of two odd operators are in c.  normal_on_x: X carries A, B and
// Y carries P, Q; otherwise mirrored (both are exact operator identities).
static std::vector<CutTerm> cut_terms(const Part &X, const Part &Y, bool normal_on_x) {
  std::vector<CutTerm> out;
  for (int i : Y.orbs) {   // a+_i S^X_i + h.c., i in Y
    Fac sx = X.op({K_S, i, -1}), cy = Y.op({K_C, i, -1});
    out.push_back({-1.0, sx, cy});                              // a+_i S^X_i = -S^X_i a+_i
    out.push_back({1.0, fac_dagger(sx), fac_dagger(cy)});       // (S^X_i)+ a_i
  }
  for (int i : X.orbs) {   // a+_i S^Y_i + h.c., i in X
    Fac cx = X.op({K_C, i, -1}), sy = Y.op({K_S, i, -1});
    out.push_back({1.0, cx, sy});
    out.push_back({-1.0, fac_dagger(cx), fac_dagger(sy)});      // (S^Y_i)+ a_i = -a_i (S^Y_i)+
  }
  const Part &Nn = normal_on_x ? X : Y;   // carries the normal pair operators
  const Part &Cc = normal_on_x ? Y : X;   // carries the complements
  auto emit = [&](double c, const Fac &n, const Fac &cpl) {
    if (normal_on_x) out.push_back({c, n, cpl}); else out.push_back({c, cpl, n});
  };
  for (size_t a = 0; a < Nn.orbs.size(); ++a)
    for (size_t b = a + 1; b < Nn.orbs.size(); ++b) {   // 1/2 sum_ik = sum_{i<k}
      int i = Nn.orbs[a], k = Nn.orbs[b];
      Fac an = Nn.op({K_A, i, k}), pc = Cc.op({K_P, i, k});
      emit(1.0, an, pc);
      emit(1.0, fac_dagger(an), fac_dagger(pc));
    }
  for (int i : Nn.orbs) for (int l : Nn.orbs) emit(1.0, Nn.op({K_B, i, l}), Cc.op({K_Q, i, l}));
  return out;
}

// Blocking rules of Appendix A3 for R = X u Y (X left of Y), products in left-to-right order.
Op2 Composite::op(const OpKey &key) const {
  Op2 out;
  const Integrals &I = *X.ints;
  Fac IX = X.op({K_I, -1, -1}), IY = Y.op({K_I, -1, -1});
  auto cre = [&](const Part &P, int i) { return P.op({K_C, i, -1}); };
  auto ann = [&](const Part &P, int i) { return fac_dagger(P.op({K_C, i, -1})); };
  switch (key.kind) {
    case K_I: tensor(out, IX, IY, 1.0); break;
    case K_C:
      if (X.has(key.i)) tensor(out, cre(X, key.i), IY, 1.0); else tensor(out, IX, cre(Y, key.i), 1.0);
      break;
    case K_A: {
      int i = key.i, k = key.k;
      if (X.has(i) && X.has(k)) tensor(out, X.op(key), IY, 1.0);
      else if (Y.has(i) && Y.has(k)) tensor(out, IX, Y.op(key), 1.0);
      else if (X.has(i)) tensor(out, cre(X, i), cre(Y, k), 1.0);
      else tensor(out, cre(X, k), cre(Y, i), -1.0);          // a+_i a+_k = -a+_k a+_i
      break;
    }
    case K_B: {
      int i = key.i, l = key.k;
      if (X.has(i) && X.has(l)) tensor(out, X.op(key), IY, 1.0);
      else if (Y.has(i) && Y.has(l)) tensor(out, IX, Y.op(key), 1.0);
      else if (X.has(i)) tensor(out, cre(X, i), ann(Y, l), 1.0);
      else tensor(out, ann(X, l), cre(Y, i), -1.0);           // a+_i a_l = -a_l a+_i
      break;
    }
    case K_S: {
      int x = key.i;
      tensor(out, X.op(key), IY, 1.0);
      tensor(out, IX, Y.op(key), 1.0);
      for (int j : Y.orbs) {
        tensor(out, X.op({K_Q, x, j}), ann(Y, j), 1.0);       // Q^X_xj a_j
        tensor(out, X.op({K_P, x, j}), cre(Y, j), 1.0);       // a+_j P^X_xj (P even)
      }
      for (int j : X.orbs) {
        tensor(out, ann(X, j), Y.op({K_Q, x, j}), 1.0);       // Q^Y_xj a_j (Q even)
        tensor(out, cre(X, j), Y.op({K_P, x, j}), 1.0);       // a+_j P^Y_xj
      }
      break;
    }
    case K_P: {
      int i = key.i, k = key.k;
      tensor(out, X.op(key), IY, 1.0);
      tensor(out, IX, Y.op(key), 1.0);
      for (int j : X.orbs) for (int l : Y.orbs) {
        double w = I.v(i, j, k, l) - I.v(i, l, k, j);
        if (w != 0.0) tensor(out, ann(X, j), ann(Y, l), -w);  // a_l a_j = -a_j a_l
      }
      break;
    }
    case K_Q: {
      int i = key.i, l = key.k;
      tensor(out, X.op(key), IY, 1.0);
      tensor(out, IX, Y.op(key), 1.0);
      for (int k : X.orbs) for (int j : Y.orbs) {
        double w1 = I.v(i, l, k, j) - I.v(i, j, k, l);
        double w2 = I.v(i, l, j, k) - I.v(i, k, j, l);
        if (w1 != 0.0) tensor(out, cre(X, k), ann(Y, j), w1);   // a+_k a_j
        if (w2 != 0.0) tensor(out, ann(X, k), cre(Y, j), -w2);  // a+_j a_k = -a_k a+_j
      }
      break;
    }
    case K_H: {
      tensor(out, X.op(key), IY, 1.0);
      tensor(out, IX, Y.op(key), 1.0);
      // the site carries the normal pair operators (it never has more orbitals than a block);
      // a vacuum block has no pair terms at all
      bool normal_on_x = X.is_site ? true : false;
      for (auto &t : cut_terms(X, Y, normal_on_x)) tensor(out, t.x, t.y, t.c);
      break;
    }
  }
  return out;
}

// ------------------------------------------------------------------ two-site H_eff terms
// Cut identity on A = (L, s1) | B = (s2, R) with A carrying the normal pair operators;
// every A-side and B-side operator expanded by the blocking rules (Appendix A3 "Two-site
// H_eff").  Terms with equal (symL, symR, site units) are merged.
std::vector<HTerm> heff_terms(const Integrals &ints, const std::vector<int> &orbsL, int site1,
                              int site2, const std::vector<int> &orbsR) {
  Part PL = make_block_part(&ints, orbsL), PR = make_block_part(&ints, orbsR);
  Part P1 = make_site_part(&ints, site1), P2 = make_site_part(&ints, site2);
  Composite A(PL, P1), B(P2, PR);
  std::vector<int> oa = A.orbs(), ob = B.orbs();

  struct KeyT { uint64_t l, r; int u; bool operator<(const KeyT &o) const {
    if (l != o.l) return l < o.l; if (r != o.r) return r < o.r; return u < o.u; } };
  std::map<KeyT, HTerm> acc;
  auto emit = [&](double c, const Op2 &a, const Op2 &b) {
    for (auto &ea : a.m) for (auto &eb : b.m) {
      const Mat4 &ma = ea.second.second, &mb = eb.second.second;
      for (int e1 = 0; e1 < 16; ++e1) {
        if (ma[e1] == 0.0) continue;
        for (int e2 = 0; e2 < 16; ++e2) {
          if (mb[e2] == 0.0) continue;
          KeyT k{ea.first, eb.first, e1 * 16 + e2};
          double val = c * ma[e1] * mb[e2];
          auto it = acc.find(k);
          if (it == acc.end())
            acc.emplace(k, HTerm{ea.second.first, eb.second.first, e1 / 4, e1 % 4, e2 / 4, e2 % 4, val});
          else it->second.c += val;
        }
      }
    }
  };
  Op2 IA = A.op({K_I, -1, -1}), IB = B.op({K_I, -1, -1});
  emit(1.0, A.op({K_H, -1, -1}), IB);
  emit(1.0, IA, B.op({K_H, -1, -1}));
  for (int i : ob) {   // a+_i S^A_i + h.c., i in B
    Op2 sa = A.op({K_S, i, -1}), cb = B.op({K_C, i, -1});
    emit(-1.0, sa, cb);
    emit(1.0, op2_dagger(sa), op2_dagger(cb));
  }
  for (int i : oa) {   // a+_i S^B_i + h.c., i in A
    Op2 ca = A.op({K_C, i, -1}), sb = B.op({K_S, i, -1});
    emit(1.0, ca, sb);
    emit(-1.0, op2_dagger(ca), op2_dagger(sb));
  }
  for (size_t a = 0; a < oa.size(); ++a)
    for (size_t b = a + 1; b < oa.size(); ++b) {
      Op2 aa = A.op({K_A, oa[a], oa[b]}), pb = B.op({K_P, oa[a], oa[b]});
      emit(1.0, aa, pb);
      emit(1.0, op2_dagger(aa), op2_dagger(pb));
    }
  for (int i : oa) for (int l : oa) emit(1.0, A.op({K_B, i, l}), B.op({K_Q, i, l}));

  std::vector<HTerm> out;
  out.reserve(acc.size());
  for (auto &e : acc) if (e.second.c != 0.0) out.push_back(e.second);
  return out;
}

// ------------------------------------------------------------------ renormalization pieces
std::vector<RPiece> renorm_pieces(const Integrals &ints, const std::vector<int> &orbs_block,
                                  int site, bool site_is_right,
                                  const std::vector<OpKey> &targets) {
  Part PB = make_block_part(&ints, orbs_block), PS = make_site_part(&ints, site);
  Composite C = site_is_right ? Composite(PB, PS) : Composite(PS, PB);
  std::vector<RPiece> out;
  for (const OpKey &t : targets) {
    Op2 o = C.op(t);
    for (auto &e : o.m)
      for (int el = 0; el < 16; ++el) {
        double c = e.second.second[el];
        if (c != 0.0) out.push_back({t, e.second.first, el / 4, el % 4, c});
      }
  }
  return out;
}

}  // namespace dmrg
