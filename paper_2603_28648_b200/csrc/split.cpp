// Split and truncate (SURVEY.md 8(a) a10, Appendix A5 "Truncation", reading s9; PAPER.md:49 truncation error,
// PAPER.md:51 fixed number of kept states / multiplets): the support step between two bonds of a sweep.  Per
// composite sector q_A of the grown block, rho = sum over the other side's blocks of psi psi^T in the packed
// (reduced, for SU(2)) basis; cyclic Jacobi eigen-decomposition on the host; the max_states largest weights over
// all sectors are kept (ties: sector label ascending, then eigen-index) and their eigenvectors form the isometry
// in the packed layout of dmrg_set_mps / dmrg_renormalize.  Not timed, FP64, host only ("host Jacobi
// is acceptable").
#include <algorithm>
#include <cmath>
#include <map>
#include <stdexcept>
#include <tuple>

#include "internal.h"

namespace dmrg {

namespace {
// Eigen-decomposition of the symmetric n x n matrix a (row-major, destroyed): eigenvalues descending in w,
// eigenvectors in the columns of v (row-major n x n).
void jacobi_eigh(std::vector<double> &a, int n, std::vector<double> &w, std::vector<double> &v) {
  v.assign((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i) v[(size_t)i * n + i] = 1.0;
  double total = 0.0;
  for (double x : a) total += x * x;
  for (int sweep = 0; sweep < 60; ++sweep) {
    double off = 0.0;
    for (int p = 0; p < n; ++p)
      for (int q = p + 1; q < n; ++q) off += a[(size_t)p * n + q] * a[(size_t)p * n + q];
    if (off <= 1e-30 * std::max(total, 1e-300)) break;
    for (int p = 0; p < n; ++p)
      for (int q = p + 1; q < n; ++q) {
        const double apq = a[(size_t)p * n + q];
        if (apq == 0.0) continue;
        const double theta = (a[(size_t)q * n + q] - a[(size_t)p * n + p]) / (2.0 * apq);
        const double t = (theta >= 0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
        const double c = 1.0 / std::sqrt(t * t + 1.0), s = t * c;
        for (int k = 0; k < n; ++k) {        // columns p, q
          const double akp = a[(size_t)k * n + p], akq = a[(size_t)k * n + q];
          a[(size_t)k * n + p] = c * akp - s * akq;
          a[(size_t)k * n + q] = s * akp + c * akq;
        }
        for (int k = 0; k < n; ++k) {        // rows p, q
          const double apk = a[(size_t)p * n + k], aqk = a[(size_t)q * n + k];
          a[(size_t)p * n + k] = c * apk - s * aqk;
          a[(size_t)q * n + k] = s * apk + c * aqk;
        }
        for (int k = 0; k < n; ++k) {
          const double vkp = v[(size_t)k * n + p], vkq = v[(size_t)k * n + q];
          v[(size_t)k * n + p] = c * vkp - s * vkq;
          v[(size_t)k * n + q] = s * vkp + c * vkq;
        }
      }
  }
  std::vector<int> order(n);
  for (int i = 0; i < n; ++i) order[i] = i;
  std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return a[(size_t)x * n + x] > a[(size_t)y * n + y]; });
  w.resize(n);
  std::vector<double> vs((size_t)n * n);
  for (int j = 0; j < n; ++j) {
    w[j] = a[(size_t)order[j] * n + order[j]];
    for (int k = 0; k < n; ++k) vs[(size_t)k * n + j] = v[(size_t)k * n + order[j]];
  }
  v.swap(vs);
}
}  // namespace

// psi: packed two-site vector of plan P (host).  grow_left: the left block absorbs site 1 (sweep to the right),
// otherwise the right block absorbs site 2.  prev: bond table of the block that grows.
void split_truncate(const HeffPlan &P, const BondTable &prev, int sym, bool grow_left, const double *psi,
                    int64_t max_states, SplitResult &out) {
  typedef std::pair<int, int> Label;                      // (N, second label) of the grown block
  struct Seg { int ip, s; int64_t dim, row0; };
  struct Sec {
    std::vector<Seg> segs;                                // sorted by (ip, s): the packed isometry order
    std::map<std::pair<int, int>, int> seg_index;
    std::map<std::tuple<int, int, int>, int64_t> col0;    // other side's composite (site, block sector, label) -> column
    int64_t rows = 0, cols = 0;
    std::vector<int> blocks;                              // psi blocks of this sector
    std::vector<double> w, v;
    std::vector<int> kept;
  };
  std::map<Label, Sec> secs;
  for (size_t bi = 0; bi < P.psi.size(); ++bi) {
    const PsiBlock &b = P.psi[bi];
    const int ip = grow_left ? b.iL : b.iR, s = grow_left ? b.s1 : b.s2;
    const Label q{prev.sec[ip].N + site_N(sym, s), grow_left ? b.SA : b.SB};
    Sec &S = secs[q];
    S.blocks.push_back((int)bi);
    if (!S.seg_index.count({ip, s})) { S.seg_index[{ip, s}] = -1; }
    auto okey = grow_left ? std::make_tuple(b.s2, b.iR, b.SB) : std::make_tuple(b.s1, b.iL, b.SA);
    if (!S.col0.count(okey)) { S.col0[okey] = S.cols; S.cols += grow_left ? b.dR : b.dL; }
  }
  struct Cand { double negw; Label q; int e; };
  std::vector<Cand> cand;
  for (auto &kv : secs) {
    Sec &S = kv.second;
    for (auto &si : S.seg_index) {                        // std::map iterates (ip, s) ascending
      si.second = (int)S.segs.size();
      S.segs.push_back(Seg{si.first.first, si.first.second, prev.sec[si.first.first].dim, S.rows});
      S.rows += prev.sec[si.first.first].dim;
    }
    std::vector<double> M((size_t)S.rows * S.cols, 0.0);
    for (int bi : S.blocks) {
      const PsiBlock &b = P.psi[bi];
      const Seg &sg = S.segs[S.seg_index[{grow_left ? b.iL : b.iR, grow_left ? b.s1 : b.s2}]];
      const int64_t c0 = S.col0[grow_left ? std::make_tuple(b.s2, b.iR, b.SB) : std::make_tuple(b.s1, b.iL, b.SA)];
      for (int64_t l = 0; l < b.dL; ++l)
        for (int64_t r = 0; r < b.dR; ++r) {
          const double x = psi[b.off + l * b.dR + r];
          if (grow_left) M[(size_t)(sg.row0 + l) * S.cols + c0 + r] = x;
          else M[(size_t)(sg.row0 + r) * S.cols + c0 + l] = x;
        }
    }
    const int n = (int)S.rows;
    std::vector<double> rho((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i)
      for (int j = i; j < n; ++j) {
        double acc = 0.0;
        for (int64_t c = 0; c < S.cols; ++c) acc += M[(size_t)i * S.cols + c] * M[(size_t)j * S.cols + c];
        rho[(size_t)i * n + j] = rho[(size_t)j * n + i] = acc;
      }
    jacobi_eigh(rho, n, S.w, S.v);
    for (int e = 0; e < n; ++e) cand.push_back(Cand{-S.w[e], kv.first, e});
  }
  std::stable_sort(cand.begin(), cand.end(), [](const Cand &x, const Cand &y) {
    if (x.negw != y.negw) return x.negw < y.negw;
    if (x.q != y.q) return x.q < y.q;
    return x.e < y.e;
  });
  out.discarded = 0.0;
  for (size_t i = 0; i < cand.size(); ++i) {
    if ((int64_t)i < max_states) secs[cand[i].q].kept.push_back(cand[i].e);
    else out.discarded += -cand[i].negw;
  }
  out.table.clear();
  int64_t off = 0;
  for (auto &kv : secs) {                                 // labels ascending
    Sec &S = kv.second;
    if (S.kept.empty()) continue;
    std::sort(S.kept.begin(), S.kept.end());
    const int64_t row[4] = {kv.first.first, kv.first.second, (int64_t)S.kept.size(), off};
    out.table.insert(out.table.end(), row, row + 4);
    off += (int64_t)S.kept.size();
  }
  const BondTable next = make_table(out.table.data(), (int64_t)out.table.size() / 4);
  int64_t total = 0;
  const std::vector<IsoBlock> blocks = iso_blocks(prev, next, sym, &total);
  out.iso.assign((size_t)total, 0.0);
  for (const IsoBlock &ib : blocks) {
    const Sector &ns = next.sec[ib.in];
    Sec &S = secs[Label{ns.N, ns.S}];
    auto it = S.seg_index.find({ib.ip, ib.s});
    if (it == S.seg_index.end()) continue;                // a composite state psi has no weight on: zero rows
    const Seg &sg = S.segs[it->second];
    const int n = (int)S.rows;
    for (int64_t r = 0; r < ib.rows; ++r)
      for (int64_t c = 0; c < ib.cols; ++c) out.iso[(size_t)(ib.off + r * ib.cols + c)] = S.v[(size_t)(sg.row0 + r) * n + S.kept[c]];
  }
}

}  // namespace dmrg
