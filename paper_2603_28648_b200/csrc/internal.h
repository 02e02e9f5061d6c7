// Internal types of the DMRG hot-path library (host side).  Not part of the ABI.
//
// The library is a small "block-sparse contraction VM": the host builds symmetry tables
// and flat job/segment descriptors (plan.cpp) from a symbolic expansion of the
// normal/complementary-operator Hamiltonian (symbolic.cpp);
// the device executes every descriptor list with one generic output-stationary grouped
// GEMM kernel (kernels.cu).  No arithmetic of the method runs on the host.
#pragma once
#include <array>
#include <cstdint>
#include <map>
#include <memory>
#include <set>
#include <string>
#include <unordered_map>
#include <vector>

namespace dmrg {

// ----------------------------------------------------------------------------- symbols
// Spin-orbital i = 2p + sigma (sigma 0 = up, 1 = down), SURVEY.md Appendix A1.
inline int spin_of(int i) { return (i & 1) ? -1 : 1; }

enum Kind { K_I = 0, K_H = 1, K_C = 2, K_S = 3, K_A = 4, K_B = 5, K_P = 6, K_Q = 7 };

typedef std::array<double, 16> Mat4;  // site operator, [s'][s] row-major, PAPER.md:41 order

struct Sym {  // block operator symbol in canonical form
  int kind, dag, i, k;   // U(1)xU(1): spin-orbital indices, dag = dagger.  SU(2): spatial orbitals, dag = tilde
  int rank = 0;          // SU(2): doubled tensor rank of A/B/P/Q symbols (0 or 2); others fixed by kind
  uint64_t key() const {
    return ((uint64_t)kind << 56) | ((uint64_t)dag << 52) | ((uint64_t)rank << 48) |
           ((uint64_t)(uint32_t)(i + 1) << 24) | (uint64_t)(uint32_t)(k + 1);
  }
  bool operator<(const Sym &o) const { return key() < o.key(); }
  bool operator==(const Sym &o) const { return key() == o.key(); }
};
struct DQ {
  int dN, dS;
  bool operator<(const DQ &o) const { return dN != o.dN ? dN < o.dN : dS < o.dS; }
  bool operator==(const DQ &o) const { return dN == o.dN && dS == o.dS; }
};
DQ sym_dq(const Sym &s);
Sym sym_dagger(const Sym &s);

typedef std::vector<std::pair<Sym, double>> LinComb;

struct Integrals {
  int L = 0;
  std::vector<double> h, V;  // L*L, L^4 (chemists' order)
  double e_core = 0;
  double t(int i, int j) const {
    return ((i ^ j) & 1) ? 0.0 : h[(size_t)(i >> 1) * L + (j >> 1)];
  }
  double v(int i, int j, int k, int l) const {
    if (((i ^ j) & 1) || ((k ^ l) & 1)) return 0.0;
    return V[(((size_t)(i >> 1) * L + (j >> 1)) * L + (k >> 1)) * L + (l >> 1)];
  }
};

struct OpKey { int kind, i, k; int rank = 0; };

// One factor of a two-part product: a lincomb of block symbols or an explicit site matrix.
struct Fac {
  bool is_site = false;
  LinComb lc;
  Mat4 m{};
};

// A part of a chain: a renormalized block (symbols) or a single site (explicit 4x4).
struct Part {
  bool is_site = false;
  int p = -1;                 // site orbital index when is_site
  std::vector<int> orbs;      // spin-orbitals, ascending
  std::vector<char> inside;   // size 2L
  const Integrals *ints = nullptr;
  bool has(int i) const { return inside[i] != 0; }
  Fac op(const OpKey &k) const;
};
Part make_site_part(const Integrals *ints, int p);
Part make_block_part(const Integrals *ints, const std::vector<int> &orbs);

// Operator on a two-part composite X (left) Y (right): sum_sym sym (x) Mat4, in left-to-right
// order.  Exactly one of X, Y is a site.  Evaluation applies the sign rule of Appendix A1.
struct Op2 {
  std::map<uint64_t, std::pair<Sym, Mat4>> m;
  void add(const Sym &s, const Mat4 &mat, double c);
};
struct Composite {
  Part X, Y;
  Composite(const Part &x, const Part &y) : X(x), Y(y) {}
  Op2 op(const OpKey &k) const;
  std::vector<int> orbs() const;
};
Op2 op2_dagger(const Op2 &o);

// One term of the two-site H_eff in left-to-right order:
//   c * symL (x) E[s1',s1] (x) E[s2',s2] (x) symR
struct HTerm {
  Sym L, R;
  int s1p, s1, s2p, s2;
  double c;
  // SU(2) only (doubled ranks): c [[L^kL x o1^k1]^kk x [o2^k2 x R^kR]^kk]^0, c includes <s1'||o1||s1><s2'||o2||s2>
  int kL = 0, k1 = 0, kk = 0, k2 = 0, kR = 0;
};
std::vector<HTerm> heff_terms(const Integrals &ints, const std::vector<int> &orbsL, int site1,
                              int site2, const std::vector<int> &orbsR);

// One piece of a new block operator (kind, i, k) after absorbing a site:
//   c * sym (x) E[s',s]   (block left of site)   or   c * E[s',s] (x) sym  (site left of block)
struct RPiece {
  OpKey target;
  Sym src;
  int sp, s;
  double c;
  int kB = 0, kS = 0, K = 0;   // SU(2): doubled ranks of the block symbol, the site operator and the product
};
// SU(2) counterparts (symbolic_su2.cpp): spatial orbitals, reduced site matrices, SURVEY.md Appendix A4
std::vector<HTerm> heff_terms_su2(const Integrals &ints, const std::vector<int> &orbsL, int site1,
                                  int site2, const std::vector<int> &orbsR);
std::vector<RPiece> renorm_pieces_su2(const Integrals &ints, const std::vector<int> &orbs_block,
                                      int site, bool site_is_right, const std::vector<OpKey> &targets);
// Wigner symbols with doubled arguments (symbolic_su2.cpp)
double wigner_cg(int j1, int m1, int j2, int m2, int J, int M);
double wigner_6j(int a, int b, int c, int d, int e, int f);
double wigner_9j(int a, int b, int c, int d, int e, int f, int g, int h, int i);
// sqrt((2K+1)(2J+1)(2j1'+1)(2j2'+1)) {j1 j2 J; k1 k2 K; j1' j2' J'}: the 9j prefactor of the product rule
double su2_f9(int j1, int j2, int J, int k1, int k2, int K, int j1p, int j2p, int Jp);
// class label (dN, second) of a symbol: second = d(2S_z) for U(1)xU(1), doubled rank for SU(2)
DQ sym_class(const Sym &s, int symmetry);
std::vector<RPiece> renorm_pieces(const Integrals &ints, const std::vector<int> &orbs_block,
                                  int site, bool site_is_right,
                                  const std::vector<OpKey> &targets);

// ------------------------------------------------------------------------- numeric tables
struct Sector { int N, S; int64_t dim, off; };
struct BondTable {
  std::vector<Sector> sec;
  std::map<std::pair<int, int>, int> index;
  int64_t total = 0;
  int find(int N, int S) const {
    auto it = index.find({N, S});
    return it == index.end() ? -1 : it->second;
  }
};
BondTable make_table(const int64_t *rows, int64_t n);

extern const int SITE_N[4];
extern const int SITE_S[4];

struct IsoBlock { int ip, s, in; int64_t rows, cols, off; };
int n_site_states(int sym);
int site_N(int sym, int s);
int site_S(int sym, int s);
std::vector<int> fuse_S(int sym, int S, int s);
std::vector<IsoBlock> iso_blocks(const BondTable &prev, const BondTable &next, int sym, int64_t *total);

// Buffer ids used by operand references; ref = (buf << 48) | element offset.
enum Buf { B_OPS_L = 0, B_OPS_R = 1, B_DER_L = 2, B_DER_R = 3, B_SCRATCH = 4, B_PSI_IN = 5,
           B_PSI_OUT = 6, B_ISO = 7, B_COEF = 8, B_NEW = 9, B_DER_TMP = 10, B_PARTIAL = 11, N_BUFS = 12 };
typedef int64_t ref_t;
inline ref_t mkref(int buf, int64_t off) { return ((int64_t)buf << 48) | off; }

// Device-consumed descriptors of the generic grouped GEMM (kernels.cu):
//   C[m][n] = colscale[n / n1] * sum_seg alpha * sum_k A[m][k] B[k][n]
//   A addr = a + m*a_ms + (k / a_kn1)*a_khi + (k % a_kn1)*a_klo
//   B addr = b + k*b_ks + (n / n1)*b_nhi + (n % n1)*b_nlo
//   C addr = c + m*c_ms + (n / n1)*c_nhi + (n % n1)*c_nlo
struct SegDesc {
  ref_t a, b;
  int64_t a_khi, b_nhi;
  int32_t K, a_ms, a_kn1, a_klo, b_ks, b_nlo;
  double alpha;
};
struct JobDesc {
  ref_t c, scale;  // scale < 0: none
  int64_t c_nhi;
  int32_t M, N, c_ms, n1, c_nlo, seg_begin, seg_end, n_iters;  // n_iters = sum_seg ceil(K / 16)
};
struct TileDesc { int32_t job, m0, n0, work; };   // work: n-tiles in this CTA's strip
struct DiagTerm {
  ref_t l, r;        // first diagonal element of the left / right operator block
  int32_t ls, rs;    // strides along the diagonal
  double f;
};
struct DiagJob { int64_t off; int32_t dL, dR, t_begin, t_end; };
// psi'[out + e] = sum_c partial[part + c * mn + e]: deterministic reduction of the stage-2 K chunks
struct ReduceJob { int64_t out, part; int32_t mn, n_chunks; };

// ---- emulated-FP64 engine (emu_seg.cuh).  A sliced operand unit (`lines` lines of K = n_members * dl digits,
// zero filled to a multiple of 32) is stored pre-tiled in the shared-memory layout of the tcgen05 operands, so that one pipeline stage
// is one contiguous bulk copy:  [line tile of R][k step of 32][slice][16-byte k chunk (2)][R rows][16 B] for R = 128 and [..][k chunk][slice][R rows][16 B] for R = 64,
// R = 128 for the left (A) operand, 64 for the right (B) operand.  Offsets are bytes at one slice (x kappa).
// The R = 128 layout above is that of the units k_emu_s1 keeps resident (s1_layout = 1).  Every other 128-row unit (the A
// operand of k_emu_seg) is stored [line tile][k step][group of 8 rows (16)][slice][k chunk (2)][8 rows][16 B], so that the
// rows that exist in a ragged tile are ONE contiguous prefix of every k step: stage 2 is HBM bound and its blocks are mostly
// narrower than 128 rows.
struct EmuSliceDesc {   // element(line, member, l) = src + member * mstride + l * lstride + line * linestride
  ref_t src;
  int64_t mstride, lstride, linestride;
  int32_t n_members, dl, line_base, lines;   // the unit's lines [line_base, line_base + lines) come from this descriptor
  int32_t dlpad, s1_layout;     // K index = member * dlpad + l (dlpad >= dl, zero filled); s1_layout: see above (R = 128 only)
  int64_t out_off;              // bytes at one slice; a unit of n lines occupies ceil(n / R) * R * ld
  int64_t tile_rows;            // R
  int64_t ld;                   // K = n_members * dlpad rounded up to a multiple of 32
  int64_t exp_off;              // index of the first line exponent (int32)
  // exponent source: bound = 0 takes the exact line maximum (two reads of the unit); bound = 1 takes the
  // Cauchy-Schwarz bound norms[psi_blk] * norms[qn_off + line] >= max |T| (one read);
  // bound = 2: the unit is written by the epilogue of the emulated stage 1 (same bound), not by the slicing kernel
  int64_t qn_off;
  int32_t psi_blk, bound;
};
struct EmuNormDesc {    // norms[out_off + line] = max_member |coef[member]| * || O_member[line][:] ||_2
  ref_t src;
  int64_t mstride, rstride, linestride, coef_off, out_off;
  int32_t n_members, dR, lines, pad;
};
struct EmuPsiDesc { int64_t off; int32_t dL, dR; };   // norms[block] = max_l || psi_block[l][:] ||_2
#ifdef __CUDACC__
#define DMRG_HD __host__ __device__
#else
#define DMRG_HD
#endif
// Performant mode (reading s21; restated by oracle/ozaki.py performant_keep): a task class
// whose magnitude bound 2^E_all lies 8 d bits below the job's reference 2^E_ref keeps kappa - d slices, at least kmin.
DMRG_HD inline int emu_keep_rule(int kappa, int kmin, int E_ref, int E_all) {
  const int d = E_ref > E_all ? (E_ref - E_all) >> 3 : 0;
  const int lim = kappa > kmin ? kappa - kmin : 0;
  return kappa - (d < lim ? d : lim);
}
constexpr int EMU_NO_REF = -(1 << 28);          // E_nz of a class without a line of non-zero exponent on either side
struct EmuSeg {         // one exponent set: rows of a sliced left unit, columns of a sliced T unit
  int64_t a_off, b_off, ea_off, eb_off;
  int32_t ksteps, keep;   // keep: slice products s + u < keep are formed when the kernel runs in performant mode (k_emu_choose)
  double alpha;
};
// rows_split = 0: C[row][n] at c + row * c_ld + (n % n1) + (n / n1) * c_nhi, scaled by scale[n / n1] (scale < 0: none)
// rows_split = 1: C[row][n] at c + (row % n1) + (row / n1) * c_nhi + n * c_ld, scaled by scale[row / n1]  (stage 1: rows are
//                 the operator lines (member, r'), columns the psi rows l, T[member][l][r'])
// fuse = 1 (stage 1 only): the epilogue also emits the INT8 slices of T for stage 2 (units of `per_piece` members at
// t_out_off + piece * piece_bytes, exponents at t_exp_off + piece * n1, K = member * dlpad + l) with the bound exponents
// norms[psi_blk] * norms[qn_off + r']; write_fp64 = 0 then skips the FP64 copy of T (no FP64 consumer).
struct EmuJob {
  ref_t c, scale; int64_t c_nhi; int32_t M, N, c_ld, n1, seg_begin, seg_end, rows_split, fuse;
  int64_t t_out_off, piece_bytes, t_exp_off, qn_off;
  int32_t per_piece, dlpad, ld_full, ld_last, n_pieces, psi_blk, write_fp64, s1_new;   // s1_new: runs in k_emu_s1 (no EmuTile)
};
struct EmuTile { int32_t job, m0, n0, work; };   // work: gang size set by the backend's schedule (0, 1: none)
// Second-generation emulated stage 1 (emu_s1.cuh): a work item is one 128-line tile of a sliced right-operator unit,
// resident in shared memory while it meets the psi rows (32 at a time) of every job that uses the unit.
struct EmuS1Item {
  int64_t a_off;                 // bytes at one slice: the line tile in the right-operator slice buffer
  int32_t ea_off, ksteps;        // first line exponent of the unit; k steps of 32 (<= s1_kres)
  int32_t m0, lines;             // first line of the tile, lines of the unit (= members * d_R')
  int32_t nt_begin, nt_end;      // EmuS1Tile range (shared by all line tiles of the unit)
  int32_t n1, pad;               // d_R': line = member * n1 + r'
};
struct EmuS1Tile {
  int64_t b_off;                 // bytes at one slice: the 32-row tile of the psi unit (all its k steps are contiguous)
  int32_t job, n0, eb_off, pad;  // stage-1 job (output addressing, exponents), first psi row, first psi row exponent
};
struct EmuPass {        // emulated part of one pass: stage-1 jobs (psi x right operators -> T), T slicing, stage-2 jobs
  std::vector<EmuSeg> segs1;
  std::vector<EmuJob> jobs1;
  std::vector<EmuTile> tiles1;
  std::vector<EmuS1Item> items1;       // jobs1 with s1_new set run in k_emu_s1 through these
  std::vector<EmuS1Tile> ntiles1;
  std::vector<EmuSliceDesc> sliceT;
  std::vector<EmuSeg> segs;
  std::vector<EmuJob> jobs;
  std::vector<EmuTile> tiles;
};

struct JobList {
  std::vector<JobDesc> jobs;
  std::vector<SegDesc> segs;
  std::vector<TileDesc> tiles;
  int64_t flops = 0;  // algorithmic 2mnk
  int tile = 32;      // CTA tile edge used by make_tiles
  void clear() { jobs.clear(); segs.clear(); tiles.clear(); flops = 0; }
};
void make_tiles(JobList &jl, int BM, int BN, int strip);

// A class of stored (or derived) block operators sharing (kind, dq): members stacked
// alpha-major per sector pair, each member block row-major [bra][ket].
struct OpBlock { int bra, ket; int64_t off; };
struct OpClass {
  int kind; DQ dq;
  std::vector<std::pair<int, int>> members;           // (i, k)
  std::map<std::pair<int, int>, int> member_index;
  std::vector<OpBlock> blocks;
  std::map<std::pair<int, int>, int> block_index;     // (bra, ket) -> idx
  int n() const { return (int)members.size(); }
};
struct DerivedClass {      // lincombs of one stored class: rows of W[n_derived][n_members]
  int cls;                 // index of the source class
  std::vector<std::vector<double>> weights;
  std::map<std::vector<double>, int> dedupe;
  std::vector<int64_t> block_off;  // per source block: offset in the derived buffer
  int64_t coef_off = 0;            // offset of W in the coefficient buffer
};
struct BlockState {
  int sym = 0;             // 0: U(1)xU(1) (spin-orbital symbols), 1: SU(2) (spatial orbitals, reduced operators)
  std::vector<int> orbs;   // spin-orbitals inside
  int n_orb = 0;           // spatial orbitals
  BondTable tab;
  std::vector<OpClass> classes;
  std::map<std::tuple<int, int, int>, int> class_index;  // (kind, dN, dS)
  int64_t elems = 0;
  void *dev = nullptr;     // device arena (doubles)
  int find_class(int kind, DQ dq) const {
    auto it = class_index.find(std::make_tuple(kind, dq.dN, dq.dS));
    return it == class_index.end() ? -1 : it->second;
  }
};
// Lay out the normal operator set {I, H, C, S, A, B} of a block.
void layout_block(BlockState &b, int L);
std::vector<OpKey> block_targets(const BlockState &b);

struct OpRef { int derived; int arr; int idx; };   // arr: class index (stored) or derived-class idx

// Resolver of symbols to operator arrays of one block, creating derived operators on demand.
struct Resolver {
  const Integrals *ints;
  const BlockState *blk;
  std::vector<DerivedClass> derived;           // one per source class that needs it
  std::map<int, int> derived_of_class;
  // flat expansion of a symbol: source class, dagger flag, weights over the class members
  bool flat(const Sym &s, int *cls, int *dag, std::vector<double> *w, int *single_idx) const;
  OpRef resolve_weights(int cls, const std::vector<double> &w);
  OpRef resolve(const Sym &s, int *dag);
  int64_t finalize(int64_t *coef_elems);       // assigns offsets; returns derived elems
  void contraction_jobs(JobList &jl, int buf_ops, int buf_der, int64_t coef_base) const;
  void coef_data(std::vector<double> &out) const;
};

static const int32_t FLAT = 1 << 30;   // n1 / kn1 value of a single-level index
static const int STRIP = 8;            // n-tiles per CTA for the short-K lists (stage 1, rotation 1, contraction)
// address of member r.idx of operator array r for the stored-orientation block (bra, ket)
bool op_addr(const Resolver &res, const OpRef &r, int buf_ops, int buf_der, int bra, int ket, ref_t *ref,
             int *cls_out);
bool consecutive(const OpRef &a, const OpRef &b);

struct Run {      // alpha-contiguous slice of a stacked group
  OpRef L, R;     // first member
  int n;
  int64_t coef_off;  // +c vector at coef_off, -c vector at coef_off + n (coefficient buffer)
  std::vector<double> c;
};
struct Group {
  int s1p, s1, s2p, s2;
  int clsL, dagL, clsR, dagR;   // class index in the block (kind via classes[cls])
  int k1 = 0, kk = 0, k2 = 0;   // SU(2): doubled ranks of the site operators and of the two coupled halves
  DQ dqL, dqR;                  // effective (after dagger)
  std::vector<Run> runs;
};

struct PsiBlock { int iL, s1, SA, s2, iR, SB; int64_t dL, dR, off; };   // SA, SB: second labels of (L,s1), (s2,R)

// Plan-time knobs (dmrg_set_option; the defaults are what bench.py times).  They choose which jobs run on the tensor
// cores in the reduced-precision modes and how the apply is cut into passes; no knob changes what is computed.
struct PlanOptions {
  int emu_mink = 128, emu_minm = 0, emu_minn = 16;         // stage-2 segment goes to tcgen05 when K, d_L', d_R' reach these
                                                           // (emu_minm = 0: chosen from the sector sizes, plan_heff_jobs.cpp)
  int emu_mink1 = 1, emu_minm1 = 1, emu_minn1 = 1;         // stage-1 job goes to tcgen05 when d_R, d_L, n_alpha d_R' reach these (every job:
                                                           // the fused T slices save more than the padding of small jobs costs, measured on configs[2..4])
  int emu_stage1 = 1;       // 0: stage 1 stays native FP64 in the reduced-precision modes
  int emu_fuse = 1;         // stage-1 epilogue emits the slices of T (0: a separate slicing pass)
  int emu_exact_exp = 0;    // 1: exact line maxima for the exponents of T (two reads) instead of the bound of reading s12b
  int emu_gang = 1;         // stage-2 tiles of one job start together (L2 reuse); 0: independent tiles
  int emu_s1new = 1;        // stage 1 on k_emu_s1 (resident operator tile); 0: on the generic k_emu_seg
  int emu_kmin = 3;         // performant mode: fewest slices a task class keeps
  int emu_kpiece = 16384;   // largest K of one emulated stage-2 segment (INT32 accumulators: 7 * 16384 * 2^14 < 2^31)
  int tile = 0;             // CTA tile edge of k_gemm_f64: 32, 48, 64; 0 = chosen from the sector sizes
  double sweep_eps = 0;     // dmrg_sweep stops when three subsequent sweep energies differ by less than this (0: off; PAPER.md:51 uses 1e-5)
  double scratch_gb = 0;    // budget for the intermediate T per pass in GB; 0 = default (32 GiB; 4 GiB of FP64 T in the tensor modes)
  int debug = 0;            // print plan statistics to stderr
};

struct HeffPlan {
  PlanOptions opt;
  std::vector<PsiBlock> psi;
  std::map<std::tuple<int, int, int, int, int, int>, int> psi_index;
  int64_t psi_len = 0;
  std::vector<Group> groups;
  Resolver resL, resR;
  JobList contractL, contractR;  // a3: derived operator build
  std::vector<JobList> stage1v, stage2v;   // a5, a6: one pair of lists per pass (T is reused between passes)
  int64_t scratch_budget = (int64_t)1 << 62, flops1 = 0, flops2 = 0;
  // emulated mode (DMRG_PREC_FP64_EMU): two-sided stage-2 segments that are large enough run on the INT8
  // tensor cores (emu[pass]); everything else stays in the FP64 lists; both meet in the split-K partial slots
  bool emu_mode = false;
  bool emu_tf32 = false;        // the tensor-core lists run as 3xTF32 (tf32_seg.cuh): same lists, exponents unused
  int kappa = 6;                // slices of the emulated mode the plan is built for (sizes the resident tile of k_emu_s1)
  std::vector<EmuSliceDesc> sliceL;      // left operators (stage-2 A operand), once per bond
  std::vector<EmuSliceDesc> sliceR;      // right operators (stage-1 B operand), once per bond
  std::vector<EmuSliceDesc> sliceP;      // psi blocks (stage-1 A operand), every apply
  std::vector<EmuPass> emu;
  std::vector<EmuNormDesc> emu_norms;
  int64_t emu_norm_elems = 0;   // psi blocks first, then the operator line norms
  int64_t emuL_bytes = 0, emuT_bytes = 0, expL_n = 0, expT_n = 0, flops_emu = 0;
  int64_t emuR_bytes = 0, emuP_bytes = 0, expR_n = 0, expP_n = 0, flops_emu1 = 0;   // bytes at one slice
  std::vector<DiagTerm> diag_terms;
  std::vector<DiagJob> diag_jobs;
  std::vector<ReduceJob> reduce;   // stage-2 split-K partial sums
  int64_t partial_elems = 0;
  std::vector<double> coef;      // host image of the coefficient buffer
  int64_t scratch_elems = 0, derL_elems = 0, derR_elems = 0;
  int64_t falg = 0;
  std::vector<int64_t> tab_psi, tab_groups, tab_counts, tab_opL, tab_opR, tab_falg_blocks;
};
// ---- split and truncate (split.cpp, row a10): host, FP64
struct SplitResult { std::vector<int64_t> table; std::vector<double> iso; double discarded = 0; };
void split_truncate(const HeffPlan &P, const BondTable &prev, int sym, bool grow_left, const double *psi,
                    int64_t max_states, SplitResult &out);

void build_heff_jobs(HeffPlan &P, const BlockState &Lb, const BlockState &Rb, int N, int twoS, int BM, int BN);
void build_heff_plan(HeffPlan &P, const Integrals &ints, const BlockState &Lb, const BlockState &Rb,
                     int site1, int site2, int N, int twoS, int BM, int BN, int64_t scratch_budget, bool emu = false,
                     bool tf32 = false, int kappa = 6, const PlanOptions *opt = nullptr);

struct RenormPlan {
  // Reduced-precision rotation (row a9 in the emulated and 3xTF32 modes): the rot1 / rot2 products as lists of the
  // tensor-core engine (emu_seg.cuh / tf32_seg.cuh), held in the emulated fields of a HeffPlan so that the backend's
  // upload / slice / run calls serve both: "stage 1" = rot1 (A: operator lines in sliceR, B: isometry columns in
  // sliceP), "stage 2" = rot2 (A: the intermediate Y in sliceL, sliced after rot1; B: isometry columns in emu[0].sliceT)
  std::shared_ptr<HeffPlan> emu;
  BlockState next;               // layout of the grown block (dev not yet allocated)
  Resolver res;
  JobList contract, rot1, rot2;
  std::vector<double> coef;
  int64_t scratch_elems = 0, der_elems = 0;
  std::vector<IsoBlock> iso;
  int64_t iso_elems = 0;
};
void build_renorm_plan(RenormPlan &P, const Integrals &ints, const BlockState &blk, int site,
                       bool site_is_right, const BondTable &new_tab, int L, int BM, int BN, bool emu = false,
                       const PlanOptions *opt = nullptr);

std::vector<int64_t> op_block_table(const BlockState &b);

}  // namespace dmrg
