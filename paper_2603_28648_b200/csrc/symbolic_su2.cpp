// Spin-adapted (SU(2)) symbolic expansion: Wigner symbols, reduced site operators, and the
// spin-adapted cut identity and blocking rules of SURVEY.md Appendix A4 (PAPER.md:51 fixes only
// that the block states are SU(2) multiplets; readings s8, s9).  All spins are doubled
// integers.  Conventions: Condon-Shortley Clebsch-Gordan coefficients; Wigner-Eckart with a bare
// CG factor, <a'j'm'|T^k_q|ajm> = <jm;kq|j'm'> <a'j'||T^k||aj>; tilde T~_m = (-1)^{k-m} (T_{-m})+.
//
// Site operators are built as explicit spherical components on the 4-dimensional site space from
// the spin-orbital definitions and reduced by Wigner-Eckart projection, so no product formula for
// same-site operators is needed.  Block operators are symbols; coupling coefficients between a
// block and a site (9j) are applied numerically by plan.cpp.
#include <algorithm>
#include <cmath>
#include <stdexcept>

#include "internal.h"

namespace dmrg {

// ------------------------------------------------------------------ Wigner symbols (Racah)
static double lfact(int n) { return std::lgamma((double)n + 1.0); }
static bool tri(int a, int b, int c) { return c >= std::abs(a - b) && c <= a + b && ((a + b + c) % 2) == 0; }

double wigner_cg(int j1, int m1, int j2, int m2, int J, int M) {
  if (m1 + m2 != M || !tri(j1, j2, J)) return 0.0;
  if (std::abs(m1) > j1 || std::abs(m2) > j2 || std::abs(M) > J) return 0.0;
  if (((j1 + m1) & 1) || ((j2 + m2) & 1) || ((J + M) & 1)) return 0.0;
  auto h = [](int x) { return x / 2; };
  double lp = std::log((double)J + 1.0) + lfact(h(J + j1 - j2)) + lfact(h(J - j1 + j2)) + lfact(h(j1 + j2 - J)) -
              lfact(h(j1 + j2 + J) + 1) + lfact(h(J + M)) + lfact(h(J - M)) + lfact(h(j1 - m1)) +
              lfact(h(j1 + m1)) + lfact(h(j2 - m2)) + lfact(h(j2 + m2));
  double s = 0.0;
  for (int k = 0;; ++k) {
    int a0 = h(j1 + j2 - J) - k, a1 = h(j1 - m1) - k, a2 = h(j2 + m2) - k;
    if (a0 < 0 || a1 < 0 || a2 < 0) break;
    int a3 = h(J - j2 + m1) + k, a4 = h(J - j1 - m2) + k;
    if (a3 < 0 || a4 < 0) continue;
    double t = std::exp(0.5 * lp - lfact(k) - lfact(a0) - lfact(a1) - lfact(a2) - lfact(a3) - lfact(a4));
    s += (k & 1) ? -t : t;
  }
  return s;
}

static double ldelta(int a, int b, int c) {   // log of the triangle coefficient, doubled arguments
  return 0.5 * (lfact((a + b - c) / 2) + lfact((a - b + c) / 2) + lfact((-a + b + c) / 2) - lfact((a + b + c) / 2 + 1));
}
double wigner_6j(int a, int b, int c, int d, int e, int f) {
  if (!tri(a, b, c) || !tri(c, d, e) || !tri(a, e, f) || !tri(b, d, f)) return 0.0;
  double lp = ldelta(a, b, c) + ldelta(c, d, e) + ldelta(a, e, f) + ldelta(b, d, f);
  int t1 = (a + b + c) / 2, t2 = (c + d + e) / 2, t3 = (a + e + f) / 2, t4 = (b + d + f) / 2;
  int u1 = (a + b + d + e) / 2, u2 = (a + c + d + f) / 2, u3 = (b + c + e + f) / 2;
  int lo = std::max(std::max(t1, t2), std::max(t3, t4)), hi = std::min(u1, std::min(u2, u3));
  double s = 0.0;
  for (int t = lo; t <= hi; ++t) {
    double v = std::exp(lp + lfact(t + 1) - lfact(t - t1) - lfact(t - t2) - lfact(t - t3) - lfact(t - t4) -
                        lfact(u1 - t) - lfact(u2 - t) - lfact(u3 - t));
    s += (t & 1) ? -v : v;
  }
  return s;
}
// {a b c; d e f; g h i} = sum_x (-1)^{2x} (2x+1) {a b c; f i x} {d e f; b x h} {g h i; x a d}
double wigner_9j(int a, int b, int c, int d, int e, int f, int g, int h, int i) {
  if (!tri(a, b, c) || !tri(d, e, f) || !tri(g, h, i) || !tri(a, d, g) || !tri(b, e, h) || !tri(c, f, i)) return 0.0;
  int lo = std::max(std::abs(a - i), std::max(std::abs(b - f), std::abs(d - h)));
  int hi = std::min(a + i, std::min(b + f, d + h));
  double s = 0.0;
  for (int x = lo; x <= hi; x += 2) {
    double v = (x + 1.0) * wigner_6j(a, b, c, f, i, x) * wigner_6j(d, e, f, b, x, h) * wigner_6j(g, h, i, x, a, d);
    s += (x & 1) ? -v : v;
  }
  return s;
}
double su2_f9(int j1, int j2, int J, int k1, int k2, int K, int j1p, int j2p, int Jp) {
  double n = wigner_9j(j1, j2, J, k1, k2, K, j1p, j2p, Jp);
  if (n == 0.0) return 0.0;
  return std::sqrt((K + 1.0) * (J + 1.0) * (j1p + 1.0) * (j2p + 1.0)) * n;
}

DQ sym_class(const Sym &s, int symmetry) {
  if (symmetry == 0) return sym_dq(s);
  int dN = 0, r = 0;
  switch (s.kind) {
    case K_I: case K_H: break;
    case K_C: dN = 1; r = 1; break;
    case K_S: dN = -1; r = 1; break;            // stored as S~ (complement of a+_x, tilde form)
    case K_A: dN = 2; r = s.rank; break;
    case K_B: dN = 0; r = s.rank; break;
    case K_P: dN = -2; r = s.rank; break;       // P~
    case K_Q: dN = 0; r = s.rank; break;        // Q~
  }
  if (s.dag) dN = -dN;
  return DQ{dN, r};
}

// ------------------------------------------------------------------ site tensors
namespace {
const int SJ[3] = {0, 1, 0};      // doubled spin of the site multiplets N = 0, 1, 2
const int SN3[3] = {0, 1, 2};
int state_of(int s, int m2) { return s == 0 ? 0 : (s == 2 ? 3 : (m2 == 1 ? 1 : 2)); }

Mat4 mzero() { Mat4 m; m.fill(0.0); return m; }
Mat4 mmul(const Mat4 &a, const Mat4 &b) {
  Mat4 c = mzero();
  for (int r = 0; r < 4; ++r) for (int k = 0; k < 4; ++k) {
    double x = a[r * 4 + k];
    if (x != 0.0) for (int q = 0; q < 4; ++q) c[r * 4 + q] += x * b[k * 4 + q];
  }
  return c;
}
Mat4 mT(const Mat4 &a) { Mat4 c; for (int r = 0; r < 4; ++r) for (int q = 0; q < 4; ++q) c[r * 4 + q] = a[q * 4 + r]; return c; }
void maxpy(Mat4 &y, double a, const Mat4 &x) { for (int e = 0; e < 16; ++e) y[e] += a * x[e]; }

struct STensor {                    // spherical tensor operator on one site: components q2 -> 4x4
  int k2 = 0;
  std::map<int, Mat4> comp;
};
STensor st_scaled(const STensor &t, double c) { STensor r = t; for (auto &e : r.comp) for (double &x : e.second) x *= c; return r; }
void st_add(STensor &y, double a, const STensor &x) {
  if (y.comp.empty()) { y.k2 = x.k2; for (int q = -x.k2; q <= x.k2; q += 2) y.comp[q] = mzero(); }
  if (y.k2 != x.k2) throw std::logic_error("st_add: rank mismatch");
  for (auto &e : x.comp) maxpy(y.comp[e.first], a, e.second);
}
STensor st_creator() {              // a+_q: q = +1/2 -> a+_up, q = -1/2 -> a+_dn (basis 0,u,d,ud; a+_d|u> = -|ud>)
  STensor t; t.k2 = 1;
  Mat4 u = mzero(), d = mzero();
  u[1 * 4 + 0] = 1.0; u[3 * 4 + 2] = 1.0;
  d[2 * 4 + 0] = 1.0; d[3 * 4 + 1] = -1.0;
  t.comp[1] = u; t.comp[-1] = d;
  return t;
}
STensor st_tilde(const STensor &t) {   // T~_m = (-1)^{k-m} (T_{-m})+
  STensor r; r.k2 = t.k2;
  for (int m = -t.k2; m <= t.k2; m += 2) {
    Mat4 x = mT(t.comp.at(-m));
    if (((t.k2 - m) / 2) & 1) for (double &v : x) v = -v;
    r.comp[m] = x;
  }
  return r;
}
STensor st_couple(const STensor &a, const STensor &b, int K2) {   // [a x b]^K on the same site
  STensor r; r.k2 = K2;
  for (int Q = -K2; Q <= K2; Q += 2) {
    Mat4 x = mzero();
    for (int q1 = -a.k2; q1 <= a.k2; q1 += 2) {
      int q2 = Q - q1;
      if (std::abs(q2) > b.k2) continue;
      double c = wigner_cg(a.k2, q1, b.k2, q2, K2, Q);
      if (c != 0.0) maxpy(x, c, mmul(a.comp.at(q1), b.comp.at(q2)));
    }
    r.comp[Q] = x;
  }
  return r;
}
STensor st_scalar(const Mat4 &m) { STensor t; t.k2 = 0; t.comp[0] = m; return t; }

// Wigner-Eckart projection to the reduced 3x3 matrix, stored in a Mat4 as [s' * 4 + s]
Mat4 st_reduce(const STensor &t) {
  Mat4 r = mzero();
  if (t.comp.empty()) return r;
  for (int sp = 0; sp < 3; ++sp) for (int s = 0; s < 3; ++s) {
    bool have = false; double val = 0.0;
    for (int q = -t.k2; q <= t.k2; q += 2) for (int m = -SJ[s]; m <= SJ[s]; m += 2) {
      int mp = m + q;
      if (std::abs(mp) > SJ[sp]) continue;
      double c = wigner_cg(SJ[s], m, t.k2, q, SJ[sp], mp);
      double x = t.comp.at(q)[state_of(sp, mp) * 4 + state_of(s, m)];
      if (std::fabs(c) < 1e-12) { if (std::fabs(x) > 1e-12) throw std::logic_error("site operator is not a tensor operator"); continue; }
      double v = x / c;
      if (have && std::fabs(v - val) > 1e-10) throw std::logic_error("site operator violates Wigner-Eckart");
      have = true; val = v;
    }
    r[sp * 4 + s] = have ? val : 0.0;
  }
  return r;
}
}  // namespace

// Reduced matrix of the site operator named by `key` on orbital t (spatial), SURVEY.md Appendix A4:
//   C = a+_t (k=1/2), A^k_tt, B^k_tt = [a+ x a~]^k, H (scalar), S~_x, P~^k_pr, Q~^k_ps (region = the site).
Mat4 su2_site_reduced(const Integrals &I, int t, const OpKey &key, int *rank2) {
  auto hh = [&](int p, int q) { return I.h[(size_t)p * I.L + q]; };
  auto vv = [&](int p, int q, int r, int s) { return I.V[(((size_t)p * I.L + q) * I.L + r) * I.L + s]; };
  STensor cr = st_creator(), an = st_tilde(cr);
  Mat4 eye = mzero();
  for (int s = 0; s < 4; ++s) eye[s * 4 + s] = 1.0;
  STensor out;
  switch (key.kind) {
    case K_I: out = st_scalar(eye); break;
    case K_C: out = cr; break;
    case K_A: out = st_couple(cr, cr, key.rank); break;
    case K_B: out = st_couple(cr, an, key.rank); break;
    case K_H: {   // h_tt n + 1/2 (tt|tt) n (n - 1): diagonal in the site basis
      Mat4 m = mzero();
      const int nocc[4] = {0, 1, 1, 2};
      for (int s = 0; s < 4; ++s) m[s * 4 + s] = hh(t, t) * nocc[s] + 0.5 * vv(t, t, t, t) * nocc[s] * (nocc[s] - 1);
      out = st_scalar(m);
      break;
    }
    case K_S: {   // S_{x sigma} = 1/2 h_xt a_{t sigma} + (xt|tt) n_t a_{t sigma};  S~_m = (-1)^{1/2-m} S_{x,-m}
      int x = key.i;
      Mat4 au = mT(cr.comp.at(1)), ad = mT(cr.comp.at(-1));
      Mat4 n = mzero();
      const int nocc[4] = {0, 1, 1, 2};
      for (int s = 0; s < 4; ++s) n[s * 4 + s] = nocc[s];
      Mat4 su = mzero(), sd = mzero();
      maxpy(su, 0.5 * hh(x, t), au); maxpy(su, vv(x, t, t, t), mmul(n, au));
      maxpy(sd, 0.5 * hh(x, t), ad); maxpy(sd, vv(x, t, t, t), mmul(n, ad));
      out.k2 = 1;
      out.comp[1] = sd;                       // m = +1/2: (-1)^0 S_{x,down}
      Mat4 neg = su; for (double &v : neg) v = -v;
      out.comp[-1] = neg;                     // m = -1/2: (-1)^1 S_{x,up}
      break;
    }
    case K_P: {   // P~^k_pr = (pt|rt) A~^k_tt (A^1_tt = 0)
      STensor a = st_tilde(st_couple(cr, cr, key.rank));
      out = st_scaled(a, vv(key.i, t, key.k, t));
      break;
    }
    case K_Q: {   // Q~^0_ps = [2(ps|tt) - (pt|ts)] B^0_tt ;  Q~^1_ps = (pt|ts) B^1_tt
      STensor b = st_couple(cr, an, key.rank);
      double w = key.rank == 0 ? 2.0 * vv(key.i, key.k, t, t) - vv(key.i, t, t, key.k) : vv(key.i, t, t, key.k);
      out = st_scaled(b, w);
      break;
    }
    default: throw std::logic_error("bad site key");
  }
  if (rank2) *rank2 = out.k2;
  return st_reduce(out);
}

// ------------------------------------------------------------------ block (x) site composites
namespace {
struct SPart {                       // a block (symbols over spatial orbitals) or a site
  bool is_site = false;
  int t = -1;
  std::vector<int> orbs;             // spatial orbitals
  std::vector<char> inside;
  const Integrals *ints = nullptr;
  bool has(int p) const { return inside[p] != 0; }
};
SPart make_part(const Integrals *I, const std::vector<int> &orbs, bool is_site) {
  SPart P; P.is_site = is_site; P.ints = I; P.orbs = orbs;
  std::sort(P.orbs.begin(), P.orbs.end());
  P.inside.assign(I->L, 0);
  for (int p : P.orbs) P.inside[p] = 1;
  if (is_site) P.t = orbs[0];
  return P;
}
struct SFac {                        // one factor: block lincomb of symbols (all of rank k2) or reduced site matrix
  bool is_site = false;
  int k2 = 0, par = 0;               // doubled rank, parity (dN mod 2)
  LinComb lc;
  Mat4 m{};
};
Sym mk(int kind, int i, int k, int rank) { Sym s{kind, 0, i, k}; s.rank = rank; return s; }
int rank_of(const OpKey &key) {
  switch (key.kind) { case K_I: case K_H: return 0; case K_C: case K_S: return 1; default: return key.rank; }
}
int par_of(int kind) { return (kind == K_C || kind == K_S) ? 1 : 0; }

SFac part_op(const SPart &P, const OpKey &key) {
  SFac f; f.is_site = P.is_site; f.k2 = rank_of(key); f.par = par_of(key.kind);
  if (P.is_site) { f.m = su2_site_reduced(*P.ints, P.t, key, nullptr); return f; }
  const bool empty = P.orbs.empty();
  const int r = key.rank, sg = (r == 2) ? -1 : 1;     // (-1)^k
  switch (key.kind) {
    case K_I: f.lc.push_back({mk(K_I, -1, -1, 0), 1.0}); break;
    case K_H: if (!empty) f.lc.push_back({mk(K_H, -1, -1, 0), 1.0}); break;
    case K_C: f.lc.push_back({mk(K_C, key.i, -1, 0), 1.0}); break;
    case K_S: if (!empty) f.lc.push_back({mk(K_S, key.i, -1, 0), 1.0}); break;
    case K_A:   // A^0_pr = A^0_rp, A^1_pr = -A^1_rp, A^1_pp = 0
      if (key.i == key.k) { if (r == 0) f.lc.push_back({mk(K_A, key.i, key.k, 0), 1.0}); }
      else if (key.i < key.k) f.lc.push_back({mk(K_A, key.i, key.k, r), 1.0});
      else f.lc.push_back({mk(K_A, key.k, key.i, r), (double)sg});
      break;
    case K_B: f.lc.push_back({mk(K_B, key.i, key.k, r), 1.0}); break;
    case K_P:   // P~^k_rp = (-1)^k P~^k_pr
      if (empty) break;
      if (key.i == key.k) { if (r == 0) f.lc.push_back({mk(K_P, key.i, key.k, 0), 1.0}); }
      else if (key.i < key.k) f.lc.push_back({mk(K_P, key.i, key.k, r), 1.0});
      else f.lc.push_back({mk(K_P, key.k, key.i, r), (double)sg});
      break;
    case K_Q: if (!empty) f.lc.push_back({mk(K_Q, key.i, key.k, r), 1.0}); break;
  }
  return f;
}
// tilde of a symbol: C, S, A, P flip the flag ((-1)^{2k} when un-flipping);  B~^k_ps = (-1)^k B^k_sp,
// Q~ likewise;  I, H are self-tilde.
std::pair<Sym, double> sym_tilde(const Sym &s) {
  Sym r = s; double c = 1.0;
  switch (s.kind) {
    case K_I: case K_H: break;
    case K_B: case K_Q: std::swap(r.i, r.k); c = (s.rank == 2) ? -1.0 : 1.0; break;
    case K_C: case K_S: r.dag = !s.dag; if (s.dag) c = -1.0; break;     // (-1)^{2 * 1/2}
    default: r.dag = !s.dag;                                            // integer rank
  }
  return {r, c};
}
Mat4 red_tilde(const Mat4 &m, int k2) {   // <j||T~||j'> = (-1)^{j'-j+k} sqrt((2j'+1)/(2j+1)) <j'||T||j>
  Mat4 r = mzero();
  for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) {
    double x = m[b * 4 + a];            // <j'=b || T || j=a>  ->  element (bra a, ket b) of the tilde
    if (x == 0.0) continue;
    int e = (SJ[b] - SJ[a] + k2) / 2;
    r[a * 4 + b] = ((e & 1) ? -1.0 : 1.0) * std::sqrt((SJ[b] + 1.0) / (SJ[a] + 1.0)) * x;
  }
  return r;
}
SFac fac_tilde(const SFac &f) {
  SFac r = f;
  if (f.is_site) { r.m = red_tilde(f.m, f.k2); return r; }
  r.lc.clear();
  for (auto &t : f.lc) { auto st = sym_tilde(t.first); r.lc.push_back({st.first, t.second * st.second}); }
  return r;
}

struct Ent { Sym sym; int kB, kS, K, par_b, par_s; Mat4 m; };
struct Op2S {                        // sum of coef [sym^kB x site^kS]^K (or site first), X-first order
  std::map<std::tuple<uint64_t, int, int>, Ent> e;
  int K = 0;
  void add(const Sym &s, int kB, int kS, int Kt, int pb, int ps, const Mat4 &m, double c) {
    if (c == 0.0) return;
    auto key = std::make_tuple(s.key(), kS, Kt);
    auto it = e.find(key);
    if (it == e.end()) { Ent n{s, kB, kS, Kt, pb, ps, mzero()}; maxpy(n.m, c, m); e.emplace(key, n); }
    else maxpy(it->second.m, c, m);
    K = Kt;
  }
};
// out += coef [x x y]^K, x on the left part; exactly one factor is the site
void couple(Op2S &out, const SFac &x, const SFac &y, int K2, double coef) {
  const SFac &b = x.is_site ? y : x, &s = x.is_site ? x : y;
  if (b.is_site || !s.is_site) throw std::logic_error("couple: need one block and one site factor");
  if (!tri(x.k2, y.k2, K2)) return;
  for (auto &t : b.lc) out.add(t.first, b.k2, s.k2, K2, b.par, s.par, s.m, coef * t.second);
}
// tilde([T x U]^K) = (-1)^{pi_T pi_U} [T~ x U~]^K  for operators on different parts
Op2S op2_tilde(const Op2S &o) {
  Op2S r;
  for (auto &kv : o.e) {
    const Ent &en = kv.second;
    auto st = sym_tilde(en.sym);
    double c = st.second * ((en.par_b && en.par_s) ? -1.0 : 1.0);
    r.add(st.first, en.kB, en.kS, en.K, en.par_b, en.par_s, red_tilde(en.m, en.kS), c);
  }
  return r;
}

struct SComposite {
  SPart X, Y;
  const Integrals &I;
  SComposite(const SPart &x, const SPart &y) : X(x), Y(y), I(*x.ints) {}
  double vv(int p, int q, int r, int s) const { return I.V[(((size_t)p * I.L + q) * I.L + r) * I.L + s]; }
  std::vector<int> orbs() const {
    std::vector<int> o = X.orbs; o.insert(o.end(), Y.orbs.begin(), Y.orbs.end());
    std::sort(o.begin(), o.end()); return o;
  }
  SFac C(const SPart &P, int p) const { return part_op(P, OpKey{K_C, p, -1, 0}); }
  SFac Ct(const SPart &P, int p) const { return fac_tilde(C(P, p)); }      // a~_p

  // spin-adapted cut identity for X | Y (Appendix A4); scalar terms [T^k x U^k]^0 in X-first order
  void cut(Op2S &out, bool normal_on_x) const {
    const double r2 = std::sqrt(2.0), r3 = std::sqrt(3.0);
    for (int x : Y.orbs) {   // -sqrt2 ([a+_x x S~^X_x]^0 + h.c.), a+_x on Y: swap factor +1
      SFac sx = part_op(X, OpKey{K_S, x, -1, 0}), cy = C(Y, x);
      couple(out, sx, cy, 0, -r2);
      couple(out, fac_tilde(sx), fac_tilde(cy), 0, +r2);     // h.c. = (-1)^{1*1} [S~~ x C~]^0
    }
    for (int y : X.orbs) {   // -sqrt2 ([a+_y x S~^Y_y]^0 + h.c.)
      SFac cx = C(X, y), sy = part_op(Y, OpKey{K_S, y, -1, 0});
      couple(out, cx, sy, 0, -r2);
      couple(out, fac_tilde(cx), fac_tilde(sy), 0, +r2);
    }
    const SPart &Nn = normal_on_x ? X : Y, &Cc = normal_on_x ? Y : X;
    auto emit = [&](const SFac &n, const SFac &c, double coef) {
      if (normal_on_x) couple(out, n, c, 0, coef); else couple(out, c, n, 0, coef);   // even operators commute
    };
    for (size_t a = 0; a < Nn.orbs.size(); ++a)
      for (size_t b = a; b < Nn.orbs.size(); ++b)
        for (int k = 0; k <= 2; k += 2) {   // 1/2 sum_{p,r} sqrt(2k+1) (A P~ + h.c.) = sum_{p<r} + 1/2 sum_{p=r}
          int p = Nn.orbs[a], r = Nn.orbs[b];
          if (p == r && k == 2) continue;
          double w = (p == r ? 0.5 : 1.0) * std::sqrt(k + 1.0);
          SFac an = part_op(Nn, OpKey{K_A, p, r, k}), pc = part_op(Cc, OpKey{K_P, p, r, k});
          emit(an, pc, w);
          emit(fac_tilde(an), fac_tilde(pc), w);
        }
    for (int p : Nn.orbs) for (int s : Nn.orbs) {
      emit(part_op(Nn, OpKey{K_B, p, s, 0}), part_op(Cc, OpKey{K_Q, p, s, 0}), 1.0);
      emit(part_op(Nn, OpKey{K_B, p, s, 2}), part_op(Cc, OpKey{K_Q, p, s, 2}), r3);
    }
  }

  Op2S op(const OpKey &key) const {
    Op2S out;
    SFac IX = part_op(X, OpKey{K_I, -1, -1, 0}), IY = part_op(Y, OpKey{K_I, -1, -1, 0});
    const int k = key.rank, sg = (k == 2) ? -1 : 1;
    switch (key.kind) {
      case K_I: couple(out, IX, IY, 0, 1.0); break;
      case K_C:
        if (X.has(key.i)) couple(out, C(X, key.i), IY, 1, 1.0); else couple(out, IX, C(Y, key.i), 1, 1.0);
        break;
      case K_A: {
        int p = key.i, r = key.k;
        if (X.has(p) && X.has(r)) couple(out, part_op(X, key), IY, k, 1.0);
        else if (Y.has(p) && Y.has(r)) couple(out, IX, part_op(Y, key), k, 1.0);
        else if (X.has(p)) couple(out, C(X, p), C(Y, r), k, 1.0);
        else couple(out, C(X, r), C(Y, p), k, sg);              // swap rule: (-1)^k
        break;
      }
      case K_B: {
        int p = key.i, s = key.k;
        if (X.has(p) && X.has(s)) couple(out, part_op(X, key), IY, k, 1.0);
        else if (Y.has(p) && Y.has(s)) couple(out, IX, part_op(Y, key), k, 1.0);
        else if (X.has(p)) couple(out, C(X, p), Ct(Y, s), k, 1.0);
        else couple(out, Ct(X, s), C(Y, p), k, sg);             // B^k_ps = (-1)^k [a~_s x a+_p]^k, s in X
        break;
      }
      case K_S: {
        int x = key.i;
        const double c0 = -1.0 / std::sqrt(2.0), c1 = std::sqrt(1.5);
        couple(out, part_op(X, key), IY, 1, 1.0);
        couple(out, IX, part_op(Y, key), 1, 1.0);
        for (int y : Y.orbs) {
          couple(out, part_op(X, OpKey{K_Q, x, y, 0}), Ct(Y, y), 1, c0);
          couple(out, part_op(X, OpKey{K_P, x, y, 0}), C(Y, y), 1, c0);     // [a+_y x P~0]: swap +1
          couple(out, part_op(X, OpKey{K_Q, x, y, 2}), Ct(Y, y), 1, c1);
          couple(out, part_op(X, OpKey{K_P, x, y, 2}), C(Y, y), 1, c1);     // -[a+_y x P~1]: swap -1
        }
        for (int q : X.orbs) {
          couple(out, Ct(X, q), part_op(Y, OpKey{K_Q, x, q, 0}), 1, c0);
          couple(out, C(X, q), part_op(Y, OpKey{K_P, x, q, 0}), 1, c0);
          couple(out, Ct(X, q), part_op(Y, OpKey{K_Q, x, q, 2}), 1, -c1);
          couple(out, C(X, q), part_op(Y, OpKey{K_P, x, q, 2}), 1, -c1);
        }
        break;
      }
      case K_P: {
        int p = key.i, r = key.k;
        couple(out, part_op(X, key), IY, k, 1.0);
        couple(out, IX, part_op(Y, key), k, 1.0);
        for (int q : X.orbs) for (int s : Y.orbs) {
          double w = vv(p, q, r, s) + sg * vv(p, s, r, q);
          if (w != 0.0) couple(out, Ct(X, q), Ct(Y, s), k, -w);            // A~^k_qs = -[a~_q x a~_s]^k
        }
        break;
      }
      case K_Q: {
        int p = key.i, s = key.k;
        couple(out, part_op(X, key), IY, k, 1.0);
        couple(out, IX, part_op(Y, key), k, 1.0);
        for (int q : X.orbs) for (int r : Y.orbs) {
          if (k == 0) {
            couple(out, C(X, q), Ct(Y, r), 0, 2.0 * vv(p, s, q, r) - vv(p, r, q, s));
            couple(out, Ct(X, q), C(Y, r), 0, 2.0 * vv(p, s, r, q) - vv(p, q, r, s));   // B^0_rq = +[a~_q x a+_r]^0
          } else {
            couple(out, C(X, q), Ct(Y, r), 2, vv(p, r, q, s));
            couple(out, Ct(X, q), C(Y, r), 2, -vv(p, q, r, s));                          // B^1_rq = -[a~_q x a+_r]^1
          }
        }
        break;
      }
      case K_H:
        couple(out, part_op(X, key), IY, 0, 1.0);
        couple(out, IX, part_op(Y, key), 0, 1.0);
        cut(out, X.is_site);           // the site carries the normal pair operators
        break;
    }
    return out;
  }
};
}  // namespace

std::vector<RPiece> renorm_pieces_su2(const Integrals &ints, const std::vector<int> &orbs_block, int site,
                                      bool site_is_right, const std::vector<OpKey> &targets) {
  SPart PB = make_part(&ints, orbs_block, false), PS = make_part(&ints, {site}, true);
  SComposite C = site_is_right ? SComposite(PB, PS) : SComposite(PS, PB);
  std::vector<RPiece> out;
  for (const OpKey &t : targets) {
    Op2S o = C.op(t);
    for (auto &kv : o.e) {
      const Ent &en = kv.second;
      for (int sp = 0; sp < 3; ++sp) for (int s = 0; s < 3; ++s) {
        double c = en.m[sp * 4 + s];
        if (c == 0.0) continue;
        RPiece p{t, en.sym, sp, s, c};
        p.kB = en.kB; p.kS = en.kS; p.K = en.K;
        out.push_back(p);
      }
    }
  }
  return out;
}

// Cut identity on A = (L, s1) | B = (s2, R), A carrying the normal pair operators.
std::vector<HTerm> heff_terms_su2(const Integrals &ints, const std::vector<int> &orbsL, int site1, int site2,
                                  const std::vector<int> &orbsR) {
  SPart PL = make_part(&ints, orbsL, false), PR = make_part(&ints, orbsR, false);
  SPart P1 = make_part(&ints, {site1}, true), P2 = make_part(&ints, {site2}, true);
  SComposite A(PL, P1), B(P2, PR);
  std::vector<int> oa = A.orbs(), ob = B.orbs();
  std::vector<HTerm> out;
  auto emit = [&](double c, const Op2S &a, const Op2S &b) {
    for (auto &ea : a.e) for (auto &eb : b.e) {
      const Ent &x = ea.second, &y = eb.second;
      if (x.K != y.K) continue;
      for (int e1 = 0; e1 < 16; ++e1) {
        if (x.m[e1] == 0.0 || (e1 & 3) == 3 || e1 >= 12) continue;
        for (int e2 = 0; e2 < 16; ++e2) {
          if (y.m[e2] == 0.0 || (e2 & 3) == 3 || e2 >= 12) continue;
          HTerm t{x.sym, y.sym, e1 / 4, e1 % 4, e2 / 4, e2 % 4, c * x.m[e1] * y.m[e2]};
          t.kL = x.kB; t.k1 = x.kS; t.kk = x.K; t.k2 = y.kS; t.kR = y.kB;
          out.push_back(t);
        }
      }
    }
  };
  const double r2 = std::sqrt(2.0), r3 = std::sqrt(3.0);
  Op2S IA = A.op(OpKey{K_I, -1, -1, 0}), IB = B.op(OpKey{K_I, -1, -1, 0});
  emit(1.0, A.op(OpKey{K_H, -1, -1, 0}), IB);
  emit(1.0, IA, B.op(OpKey{K_H, -1, -1, 0}));
  for (int x : ob) {
    Op2S sa = A.op(OpKey{K_S, x, -1, 0}), cb = B.op(OpKey{K_C, x, -1, 0});
    emit(-r2, sa, cb);
    emit(+r2, op2_tilde(sa), op2_tilde(cb));
  }
  for (int y : oa) {
    Op2S ca = A.op(OpKey{K_C, y, -1, 0}), sb = B.op(OpKey{K_S, y, -1, 0});
    emit(-r2, ca, sb);
    emit(+r2, op2_tilde(ca), op2_tilde(sb));
  }
  for (size_t a = 0; a < oa.size(); ++a)
    for (size_t b = a; b < oa.size(); ++b)
      for (int k = 0; k <= 2; k += 2) {
        int p = oa[a], r = oa[b];
        if (p == r && k == 2) continue;
        double w = (p == r ? 0.5 : 1.0) * std::sqrt(k + 1.0);
        Op2S aa = A.op(OpKey{K_A, p, r, k}), pb = B.op(OpKey{K_P, p, r, k});
        emit(w, aa, pb);
        emit(w, op2_tilde(aa), op2_tilde(pb));
      }
  for (int p : oa) for (int s : oa) {
    emit(1.0, A.op(OpKey{K_B, p, s, 0}), B.op(OpKey{K_Q, p, s, 0}));
    emit(r3, A.op(OpKey{K_B, p, s, 2}), B.op(OpKey{K_Q, p, s, 2}));
  }
  return out;
}

}  // namespace dmrg
