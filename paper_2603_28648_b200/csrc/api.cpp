// C ABI of include/dmrg.h: context, call-order checks, memory ownership, and the host loops
// that walk the plans (dmrg_build_env, dmrg_davidson_step).  All arithmetic runs in kernels.cu.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <new>
#include <stdexcept>

#include "../../include/dmrg.h"
#include "backend.h"

using namespace dmrg;

namespace {
struct StateError : std::runtime_error { using std::runtime_error::runtime_error; };
struct Unsupported : std::runtime_error { using std::runtime_error::runtime_error; };
constexpr int MAX_DAVIDSON = 32;  // MAX_BASIS of kernels.cu
}  // namespace

struct dmrg_ctx {
  std::unique_ptr<Backend> be;   // null for a planning context
  std::string err;
  Integrals ints;
  int L = 0, N = 0, twoS = 0, sym = 0, D = 0;
  PlanOptions opt;               // dmrg_set_option
  bool plan_stale = false;       // an option changed after the plan was built: rebuilt at the next use
  bool have_ints = false, have_mps = false, env_ready = false, plan_ready = false, timing = false;
  int bond = 0;
  std::vector<BondTable> ltab, rtab;
  std::vector<void *> liso, riso;          // device copies of the isometries
  BlockState left, right;
  HeffPlan plan;
  DevJobList d_contractL, d_contractR;
  std::vector<DevJobList> d_stage1, d_stage2;   // one pair per pass
  DevDiag d_diag;
  DevReduce d_reduce;
  DevEmu d_emu;                  // emulated stage 2 (plan.emu_mode): descriptors, slice planes, exponents
  int emu_kappa = 0;             // slices the current plan was prepared for (0: native FP64 plan)
  bool performant = false;       // the current call runs DMRG_PREC_FP64_EMU_PERF (set by the H_eff entry points)
  void *partial = nullptr;
  void *derL = nullptr, *derR = nullptr, *scratch = nullptr, *coef = nullptr;
  void *psi_a = nullptr, *psi_b = nullptr;  // staging for the host-buffer apply
  void *dav = nullptr; int64_t dav_elems = 0;
  std::vector<int64_t> tab_bondL, tab_bondR, tab_isoL, tab_isoR, tab_falg;
  double ms1 = 0, ms2 = 0, ms_slice = 0, ms_int8 = 0, ms_s1_tensor = 0;
  SplitResult split;              // last dmrg_split_truncate
  // dmrg_sweep: device-resident stacks of left / right blocks (index = number of absorbed sites); while a sweep
  // runs, `left` / `right` alias stack entries and must not be released through drop_env
  std::vector<BlockState> lstack, rstack;
  bool env_borrowed = false;

  void drop_plan() {
    if (be) {
      be->free_jobs(d_contractL); be->free_jobs(d_contractR);
      for (auto &j : d_stage1) be->free_jobs(j);
      for (auto &j : d_stage2) be->free_jobs(j);
      be->free_diag(d_diag);
      be->free_reduce(d_reduce);
      be->free_emu(d_emu);
      be->release(partial);
      be->release(derL); be->release(derR); be->release(scratch); be->release(coef);
      be->release(psi_a); be->release(psi_b); be->release(dav);
    }
    derL = derR = scratch = coef = psi_a = psi_b = dav = partial = nullptr;
    dav_elems = 0;
    d_stage1.clear(); d_stage2.clear();
    plan = HeffPlan();
    plan_ready = false; emu_kappa = 0;
  }
  void drop_env() {
    drop_plan();
    if (be && !env_borrowed) { be->release(left.dev); be->release(right.dev); }
    left = BlockState(); right = BlockState();
    env_borrowed = false;
    env_ready = false;
  }
  void drop_stacks() {
    if (env_borrowed) { left = BlockState(); right = BlockState(); env_borrowed = false; env_ready = false; }
    if (be) { for (auto &b : lstack) be->release(b.dev); for (auto &b : rstack) be->release(b.dev); }
    lstack.clear(); rstack.clear();
  }
  void drop_mps() {
    drop_plan();
    drop_stacks();
    drop_env();
    if (be) { for (void *p : liso) be->release(p); for (void *p : riso) be->release(p); }
    liso.clear(); riso.clear(); ltab.clear(); rtab.clear();
    have_mps = false;
  }
  ~dmrg_ctx() { drop_mps(); }
};

#define GUARD_BEGIN                                                   \
  if (!ctx) return DMRG_EINVAL;                                       \
  try {
#define GUARD_END                                                     \
  }                                                                   \
  catch (const StateError &e) { ctx->err = e.what(); return DMRG_ESTATE; }          \
  catch (const Unsupported &e) { ctx->err = e.what(); return DMRG_EUNSUPPORTED; }   \
  catch (const std::invalid_argument &e) { ctx->err = e.what(); return DMRG_EINVAL; } \
  catch (const std::bad_alloc &) { ctx->err = "out of memory"; return DMRG_ENOMEM; }  \
  catch (const std::exception &e) {                                   \
    ctx->err = e.what();                                              \
    return std::strncmp(e.what(), "CUDA", 4) == 0 ? DMRG_ECUDA : DMRG_EINVAL;       \
  }                                                                   \
  return DMRG_OK;

// Tile edge for a plan whose largest sector dimension is `maxdim`: small sectors waste less on small
// tiles, large ones get more MMAs per issued instruction on large tiles (profiles/r1_summary.md).
static int pick_tile(const dmrg_ctx *ctx, int64_t maxdim) {
  if (ctx->opt.tile) return ctx->opt.tile;
  return maxdim >= 96 ? 64 : (maxdim >= 40 ? 48 : 32);
}
static int64_t max_dim(const BondTable &t) {
  int64_t m = 1;
  for (const Sector &s : t.sec) m = std::max(m, s.dim);
  return m;
}

static void need_gpu(dmrg_ctx *ctx) {
  if (!ctx->be) throw Unsupported("planning context: no sm_100a device bound, compute calls are unavailable "
                                  "(there is no CPU fallback)");
  ctx->be->make_current();       // every compute entry runs on the context's device, whatever the caller's current one is
}
// Returns the plan variant the mode needs: 0 = native FP64, 2..7 = emulated FP64 with that many INT8 slices,
// 8 = 3xTF32 (the value is also the bytes per sliced element).
static int check_precision(int precision, int slices = 0) {
  if (precision == DMRG_PREC_FP64) return 0;
  if (precision == DMRG_PREC_FP64_EMU || precision == DMRG_PREC_FP64_EMU_PERF) {     // performant: same plan and slices,
    if (slices == 0) return 6;                                                       // fewer products per task class             // Appendix A6 default (kappa = 6)
    if (slices < 2 || slices > 7) throw std::invalid_argument("slices must be 0 (default 6) or in [2, 7]");
    return slices;
  }
  if (precision == DMRG_PREC_TF32X3) return 8;       // 8 bytes per element (hi + lo): the 3xTF32 lists
  throw std::invalid_argument("unknown precision mode");
}

static BlockState vacuum_block(dmrg_ctx *ctx, const BondTable &tab) {
  BlockState b;
  b.sym = ctx->sym;
  b.tab = tab;
  if (tab.sec.size() != 1 || tab.sec[0].N != 0 || tab.sec[0].S != 0 || tab.sec[0].dim != 1)
    throw std::invalid_argument("table of the empty block must be the single row (0, 0, 1, 0)");
  layout_block(b, ctx->L);
  if (ctx->be) {
    b.dev = ctx->be->alloc(sizeof(double) * b.elems);
    double one = 1.0;
    ctx->be->upload(b.dev, &one, sizeof(double));
    ctx->be->sync();
  }
  return b;
}

// One renormalization step on the device: contraction (a3) -> rot1 -> rot2 (a9).
// kappa: 0 = native FP64 (DMMA); 2..7 = the two rotation products on the INT8 tensor cores with that many slices;
// 8 = 3xTF32.  The contracted-operator build (a3) is native FP64 in every mode.
static void renorm_step(dmrg_ctx *ctx, BlockState &blk, int site, bool site_is_right, const BondTable &new_tab,
                        const void *iso_dev, bool keep_old = false, int kappa = 0) {
  Backend &be = *ctx->be;
  RenormPlan P;
  build_renorm_plan(P, ctx->ints, blk, site, site_is_right, new_tab, ctx->L,
                    pick_tile(ctx, std::max(max_dim(blk.tab), max_dim(new_tab))),
                    pick_tile(ctx, std::max(max_dim(blk.tab), max_dim(new_tab))), kappa != 0, &ctx->opt);
  void *nw = nullptr, *der = nullptr, *scr = nullptr, *cf = nullptr;
  DevJobList jc, j1, j2;
  DevEmu de;
  try {
    nw = be.alloc(sizeof(double) * P.next.elems);
    der = be.alloc(sizeof(double) * P.der_elems);
    scr = be.alloc(sizeof(double) * P.scratch_elems);
    cf = be.alloc(sizeof(double) * P.coef.size());
    be.zero(nw, sizeof(double) * P.next.elems);
    be.upload(cf, P.coef.data(), sizeof(double) * P.coef.size());
    be.upload_jobs(P.contract, jc, 0);
    be.upload_jobs(P.rot1, j1, 1);
    be.upload_jobs(P.rot2, j2, 2);
    BufTable bt{};
    bt.p[site_is_right ? B_OPS_L : B_OPS_R] = (double *)blk.dev;
    bt.p[B_DER_TMP] = (double *)der; bt.p[B_SCRATCH] = (double *)scr; bt.p[B_ISO] = (double *)iso_dev;
    bt.p[B_COEF] = (double *)cf; bt.p[B_NEW] = (double *)nw;
    be.run_jobs(jc, bt);
    if (kappa == 0) {
      be.run_jobs(j1, bt);
      be.run_jobs(j2, bt);
    } else {
      be.upload_emu(*P.emu, kappa, de);
      be.run_emu_slice(de, EMU_SLICE_R, bt);        // source operators (stored and contracted), lines (alpha, l')
      be.run_emu_slice(de, EMU_SLICE_PSI, bt);      // isometry columns for rot1
      be.run_emu_stage(de, 0, 1, bt);               // rot1: Y = c O X_ket
      be.run_emu_slice(de, EMU_SLICE_L, bt);        // Y, lines (alpha, a)
      be.run_emu_slice(de, 0, bt);                  // isometry columns for rot2
      be.run_emu_stage(de, 0, 2, bt);               // rot2: O' += G X_bra^T Y
    }
    be.sync();
  } catch (...) {
    be.free_emu(de);
    be.free_jobs(jc); be.free_jobs(j1); be.free_jobs(j2);
    be.release(nw); be.release(der); be.release(scr); be.release(cf);
    throw;
  }
  be.free_emu(de);
  be.free_jobs(jc); be.free_jobs(j1); be.free_jobs(j2);
  be.release(der); be.release(scr); be.release(cf);
  if (!keep_old) be.release(blk.dev);        // the sweep driver keeps every block of both stacks
  blk = P.next;
  blk.dev = nw;
}

static std::vector<int64_t> table_rows(const BondTable &t) {
  std::vector<int64_t> r;
  for (const Sector &s : t.sec) { r.push_back(s.N); r.push_back(s.S); r.push_back(s.dim); r.push_back(s.off); }
  return r;
}
static std::vector<int64_t> iso_rows(const std::vector<IsoBlock> &v) {
  std::vector<int64_t> r;
  for (const IsoBlock &b : v) { int64_t row[6] = {b.ip, b.s, b.in, b.rows, b.cols, b.off}; r.insert(r.end(), row, row + 6); }
  return r;
}

// elements of the intermediate T per pass: 32 GiB by default, 4 GiB of FP64 T in the tensor-core modes (most of T is
// kept as slices there), or the option scratch_gb
static int64_t scratch_budget(const dmrg_ctx *ctx, int kappa) {
  const int64_t dflt = (int64_t)4 << 30;
  const int64_t b = ctx->opt.scratch_gb > 0 ? (int64_t)(ctx->opt.scratch_gb * 1e9 / 8) : dflt;
  return kappa ? std::min<int64_t>(b, (int64_t)1 << 32) : b;
}
static void prepare_heff(dmrg_ctx *ctx, int kappa = 0) {
  ctx->drop_plan();
  HeffPlan &P = ctx->plan;
  build_heff_plan(P, ctx->ints, ctx->left, ctx->right, ctx->bond, ctx->bond + 1, ctx->N, ctx->twoS,
                  pick_tile(ctx, std::max(max_dim(ctx->left.tab), max_dim(ctx->right.tab))),
                  pick_tile(ctx, std::max(max_dim(ctx->left.tab), max_dim(ctx->right.tab))), scratch_budget(ctx, kappa), kappa != 0, kappa == 8, kappa ? kappa : 6, &ctx->opt);
  ctx->plan_stale = false;
  ctx->tab_bondL = table_rows(ctx->left.tab);
  ctx->tab_bondR = table_rows(ctx->right.tab);
  ctx->tab_falg = {P.falg};
  ctx->tab_isoL.clear(); ctx->tab_isoR.clear();
  if (ctx->bond >= 1) ctx->tab_isoL = iso_rows(iso_blocks(ctx->ltab[ctx->bond - 1], ctx->ltab[ctx->bond], ctx->sym, nullptr));
  int nr = (int)ctx->rtab.size() - 1;
  if (nr >= 1) ctx->tab_isoR = iso_rows(iso_blocks(ctx->rtab[nr - 1], ctx->rtab[nr], ctx->sym, nullptr));
  if (ctx->be) {
    Backend &be = *ctx->be;
    ctx->derL = be.alloc(sizeof(double) * P.derL_elems);
    ctx->derR = be.alloc(sizeof(double) * P.derR_elems);
    ctx->scratch = be.alloc(sizeof(double) * P.scratch_elems);
    ctx->coef = be.alloc(sizeof(double) * P.coef.size());
    be.upload(ctx->coef, P.coef.data(), sizeof(double) * P.coef.size());
    be.upload_jobs(P.contractL, ctx->d_contractL, 0);
    be.upload_jobs(P.contractR, ctx->d_contractR, 0);
    ctx->d_stage1.resize(P.stage1v.size());
    ctx->d_stage2.resize(P.stage2v.size());
    for (size_t p = 0; p < P.stage1v.size(); ++p) {
      be.upload_jobs(P.stage1v[p], ctx->d_stage1[p], 3);
      be.upload_jobs(P.stage2v[p], ctx->d_stage2[p], 4);
    }
    be.upload_diag(P.diag_jobs, P.diag_terms, ctx->d_diag);
    be.upload_reduce(P.reduce, ctx->d_reduce);
    ctx->partial = be.alloc(sizeof(double) * P.partial_elems);
    BufTable bt{};
    bt.p[B_OPS_L] = (double *)ctx->left.dev; bt.p[B_OPS_R] = (double *)ctx->right.dev;
    bt.p[B_DER_L] = (double *)ctx->derL; bt.p[B_DER_R] = (double *)ctx->derR; bt.p[B_COEF] = (double *)ctx->coef;
    be.run_jobs(ctx->d_contractL, bt);
    be.run_jobs(ctx->d_contractR, bt);
    if (kappa) {             // slice-and-pack of the left operators, once per bond (row a4)
      be.upload_emu(P, kappa, ctx->d_emu);
      be.run_emu_slice(ctx->d_emu, EMU_SLICE_L, bt);
      be.run_emu_slice(ctx->d_emu, EMU_SLICE_R, bt);
      be.run_emu_norms(ctx->d_emu, -1, bt);
    }
    be.sync();
  }
  ctx->emu_kappa = kappa;
  ctx->plan_ready = true;
}

// The plan depends on the precision mode (which segments run emulated): re-plan when the mode changes.
static void ensure_plan(dmrg_ctx *ctx, int kappa) {
  if (ctx->plan_ready && (ctx->emu_kappa != kappa || ctx->plan_stale)) prepare_heff(ctx, kappa);
}

static BufTable heff_bufs(dmrg_ctx *ctx, const double *in, double *out) {
  BufTable bt{};
  bt.p[B_OPS_L] = (double *)ctx->left.dev; bt.p[B_OPS_R] = (double *)ctx->right.dev;
  bt.p[B_DER_L] = (double *)ctx->derL; bt.p[B_DER_R] = (double *)ctx->derR;
  bt.p[B_SCRATCH] = (double *)ctx->scratch; bt.p[B_COEF] = (double *)ctx->coef;
  bt.p[B_PSI_IN] = const_cast<double *>(in); bt.p[B_PSI_OUT] = out; bt.p[B_PARTIAL] = (double *)ctx->partial;
  return bt;
}
static void heff_apply(dmrg_ctx *ctx, const double *in, double *out) {
  BufTable bt = heff_bufs(ctx, in, out);
  if (ctx->timing) { ctx->ms1 = 0; ctx->ms2 = 0; ctx->ms_slice = 0; ctx->ms_int8 = 0; ctx->ms_s1_tensor = 0; }
  const size_t np = ctx->d_stage1.size();
  const bool perf = ctx->performant && ctx->emu_kappa >= 2 && ctx->emu_kappa <= 7;
  if (perf) ctx->be->reset_emu_products(ctx->d_emu);
  if (ctx->emu_kappa) {        // per apply: psi line norms (bound exponents of T) and the psi slices of stage 1
    ctx->be->run_emu_norms(ctx->d_emu, 0, bt);
    ctx->be->run_emu_slice(ctx->d_emu, EMU_SLICE_PSI, bt);
  }
  for (size_t p = 0; p < np; ++p) {
    if (ctx->timing) ctx->be->timer_mark(0);
    ctx->be->run_jobs(ctx->d_stage1[p], bt);
    if (ctx->timing) ctx->be->timer_mark(8);
    if (ctx->emu_kappa) ctx->be->run_emu_stage(ctx->d_emu, (int)p, 1, bt);
    if (ctx->timing) ctx->be->timer_mark(1);
    ctx->be->run_jobs(ctx->d_stage2[p], bt);
    if (ctx->emu_kappa) {
      if (ctx->timing) ctx->be->timer_mark(6);
      ctx->be->run_emu_slice(ctx->d_emu, (int)p, bt);
      if (perf) ctx->be->run_emu_choose(ctx->d_emu, (int)p, ctx->opt.emu_kmin);     // slice products per task class (reading s21)
      if (ctx->timing) ctx->be->timer_mark(7);
      ctx->be->run_emu_stage(ctx->d_emu, (int)p, 2, bt, perf);
      if (ctx->timing) ctx->be->timer_mark(3);
    }
    if (p + 1 == np) ctx->be->run_reduce(ctx->d_reduce, (const double *)ctx->partial, out);
    if (ctx->timing) {      // timing mode synchronises after every pass
      ctx->be->timer_mark(2);
      ctx->ms1 += ctx->be->timer_ms(0, 1);
      ctx->ms2 += ctx->be->timer_ms(1, 2);
      if (ctx->emu_kappa) {
        ctx->ms_slice += ctx->be->timer_ms(6, 7); ctx->ms_int8 += ctx->be->timer_ms(7, 3);
        ctx->ms_s1_tensor += ctx->be->timer_ms(8, 1);
      }
    }
  }
}

// Davidson iterations on the current plan (a7 + a8 around a5/a6); psi is overwritten by the normalised Ritz vector
static int davidson_run(dmrg_ctx *ctx, double *psi, int n_iter, double tol, double *theta_host, double *resid_host) {
  Backend &be = *ctx->be;
  const int64_t n = ctx->plan.psi_len;
  n_iter = (int)std::min<int64_t>(n_iter, n);          // the basis cannot outgrow the space
  const int mmax = n_iter;
  // workspace: V[mmax], W[mmax], x, r, t, diag, then small scalars
  const int64_t small = (int64_t)mmax * mmax + 6 * mmax + 8;
  const int64_t need = (2 * (int64_t)mmax + 4) * n + small;
  if (ctx->dav_elems < need) {
    be.release(ctx->dav);
    ctx->dav = nullptr; ctx->dav_elems = 0;
    ctx->dav = be.alloc(sizeof(double) * need);
    ctx->dav_elems = need;
  }
  double *V = (double *)ctx->dav, *W = V + (int64_t)mmax * n, *x = W + (int64_t)mmax * n, *r = x + n, *t = r + n,
         *dg = t + n, *G = dg + n, *col = G + mmax * mmax, *y = col + mmax, *theta = y + mmax,
         *res2 = theta + mmax, *cproj = res2 + mmax, *nrm2 = cproj + mmax;
  be.zero(G, sizeof(double) * small);
  BufTable bt = heff_bufs(ctx, nullptr, nullptr);
  be.run_diag(ctx->d_diag, bt, dg);
  be.dots(psi, n, 1, psi, n, nrm2);
  be.scale_inv_norm(psi, nrm2, V, n);
  int done = 0;
  for (int it = 0; it < n_iter; ++it) {
    const int m = it + 1;
    heff_apply(ctx, V + (int64_t)it * n, W + (int64_t)it * n);
    be.dots(V, n, m, W + (int64_t)it * n, n, col);
    be.davidson_small(G, mmax, m, col, y, theta + it);
    be.ritz_residual(V, W, n, m, n, y, theta + it, x, r);
    be.dots(r, n, 1, r, n, res2 + it);
    done = m;
    if (it == n_iter - 1) break;
    if (tol > 0) {
      double r2;
      be.download(&r2, res2 + it, sizeof(double));
      if (std::sqrt(r2) < tol) break;
    }
    be.precondition(r, dg, theta + it, t, n);
    for (int pass = 0; pass < 2; ++pass) {
      be.dots(V, n, m, t, n, cproj);
      be.subtract_projection(V, n, m, cproj, t, n);
    }
    be.dots(t, n, 1, t, n, nrm2);
    {   // c6: the expansion vector vanished (exact eigenvector, exhausted space): stop, as oracle/davidson.py does
      double t2;
      be.download(&t2, nrm2, sizeof(double));
      if (!(std::sqrt(std::max(0.0, t2)) >= 1e-14)) break;
    }
    be.scale_inv_norm(t, nrm2, V + (int64_t)m * n, n);
  }
  be.dots(x, n, 1, x, n, nrm2);
  be.scale_inv_norm(x, nrm2, psi, n);
  std::vector<double> th(done), r2(done);
  be.download(th.data(), theta, sizeof(double) * done);
  be.download(r2.data(), res2, sizeof(double) * done);
  for (int i = 0; i < done; ++i) { theta_host[i] = th[i]; resid_host[i] = std::sqrt(std::max(0.0, r2[i])); }
  return done;
}

extern "C" {

int dmrg_create(dmrg_ctx **out, int device, void *cuda_stream) {
  if (!out) return DMRG_EINVAL;
  *out = nullptr;
  dmrg_ctx *c = new (std::nothrow) dmrg_ctx();
  if (!c) return DMRG_ENOMEM;
  if (device >= 0) {
    std::string err;
    Backend *b = make_cuda_backend(device, cuda_stream, &err);
    if (!b) { delete c; return DMRG_EUNSUPPORTED; }
    c->be.reset(b);
  }
  *out = c;
  return DMRG_OK;
}

int dmrg_set_option(dmrg_ctx *ctx, const char *key, double value) {
  GUARD_BEGIN
  if (!key) throw std::invalid_argument("dmrg_set_option: null key");
  PlanOptions &o = ctx->opt;
  const std::string k = key;
  const int iv = (int)value;
  struct { const char *name; int *field; int lo, hi; } ints[] = {
      {"emu_mink", &o.emu_mink, 1, 1 << 30}, {"emu_minm", &o.emu_minm, 0, 1 << 30}, {"emu_minn", &o.emu_minn, 1, 1 << 30},
      {"emu_mink1", &o.emu_mink1, 1, 1 << 30}, {"emu_minm1", &o.emu_minm1, 1, 1 << 30}, {"emu_minn1", &o.emu_minn1, 1, 1 << 30},
      {"emu_stage1", &o.emu_stage1, 0, 1}, {"emu_fuse", &o.emu_fuse, 0, 1}, {"emu_exact_exp", &o.emu_exact_exp, 0, 1},
      {"emu_gang", &o.emu_gang, 0, 1}, {"emu_kpiece", &o.emu_kpiece, 32, 16384}, {"emu_kmin", &o.emu_kmin, 1, 7}, {"emu_s1new", &o.emu_s1new, 0, 1}, {"debug", &o.debug, 0, 1}};
  bool found = false;
  for (auto &e : ints)
    if (k == e.name) {
      if (value != (double)iv || iv < e.lo || iv > e.hi) throw std::invalid_argument("dmrg_set_option: value out of range for " + k);
      *e.field = iv; found = true;
    }
  if (k == "tile") {
    if (!(iv == 0 || iv == 32 || iv == 48 || iv == 64) || value != (double)iv) throw std::invalid_argument("dmrg_set_option: tile must be 0, 32, 48 or 64");
    o.tile = iv; found = true;
  } else if (k == "sweep_eps") {
    if (!(value >= 0)) throw std::invalid_argument("dmrg_set_option: sweep_eps must be >= 0");
    o.sweep_eps = value; found = true;
  } else if (k == "scratch_gb") {
    if (!(value >= 0)) throw std::invalid_argument("dmrg_set_option: scratch_gb must be >= 0");
    o.scratch_gb = value; found = true;
  }
  if (!found) throw std::invalid_argument("dmrg_set_option: unknown option '" + k + "'");
  ctx->plan_stale = true;
  GUARD_END
}

int dmrg_destroy(dmrg_ctx *ctx) {
  if (!ctx) return DMRG_EINVAL;
  delete ctx;
  return DMRG_OK;
}

const char *dmrg_last_error(dmrg_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int dmrg_init_integrals(dmrg_ctx *ctx, int L, const double *h, const double *V, const double *chol, int n_chol,
                        double e_core, int N, int twoS, int symmetry, int D) {
  GUARD_BEGIN
  if (L < 2 || L > 512 || !h || (!V && !(chol && n_chol > 0)) || N < 0 || N > 2 * L || D < 1)
    throw std::invalid_argument("dmrg_init_integrals: bad arguments");
  if (symmetry != DMRG_SYM_U1U1 && symmetry != DMRG_SYM_SU2) throw std::invalid_argument("unknown symmetry");
  if ((N + twoS) % 2 != 0 || std::abs(twoS) > N) throw std::invalid_argument("N and 2S (2S_z) are incompatible");
  if (symmetry == DMRG_SYM_SU2 && twoS < 0) throw std::invalid_argument("2S must be non-negative");
  ctx->drop_mps();
  Integrals &I = ctx->ints;
  I.L = L; I.e_core = e_core;
  I.h.assign(h, h + (size_t)L * L);
  size_t L2 = (size_t)L * L;
  I.V.assign(L2 * L2, 0.0);
  if (V) {
    std::copy(V, V + L2 * L2, I.V.begin());
  } else {   // input marshalling only: V_ijkl = sum_c B^c_ij B^c_kl
    for (int c = 0; c < n_chol; ++c) {
      const double *B = chol + (size_t)c * L2;
      for (size_t ij = 0; ij < L2; ++ij) {
        double b = B[ij];
        if (b == 0.0) continue;
        double *row = &I.V[ij * L2];
        for (size_t kl = 0; kl < L2; ++kl) row[kl] += b * B[kl];
      }
    }
  }
  ctx->L = L; ctx->N = N; ctx->twoS = twoS; ctx->sym = symmetry; ctx->D = D;
  ctx->have_ints = true;
  GUARD_END
}

int dmrg_set_mps(dmrg_ctx *ctx, int bond, const int64_t *const *left_tables, const int64_t *left_rows,
                 const double *const *left_iso, const int64_t *const *right_tables, const int64_t *right_rows,
                 const double *const *right_iso, int on_device) {
  GUARD_BEGIN
  if (!ctx->have_ints) throw StateError("dmrg_set_mps before dmrg_init_integrals");
  if (bond < 0 || bond > ctx->L - 2 || !left_tables || !left_rows || !right_tables || !right_rows)
    throw std::invalid_argument("dmrg_set_mps: bad arguments");
  ctx->drop_mps();
  ctx->bond = bond;
  int nl = bond, nr = ctx->L - bond - 2;
  for (int m = 0; m <= nl; ++m) ctx->ltab.push_back(make_table(left_tables[m], left_rows[m]));
  for (int m = 0; m <= nr; ++m) ctx->rtab.push_back(make_table(right_tables[m], right_rows[m]));
  if (ctx->be) {
    if ((nl > 0 && !left_iso) || (nr > 0 && !right_iso)) throw std::invalid_argument("dmrg_set_mps: missing isometries");
    auto take = [&](const std::vector<BondTable> &tabs, const double *const *iso, int n, std::vector<void *> &out) {
      for (int m = 0; m < n; ++m) {
        int64_t tot = 0;
        iso_blocks(tabs[m], tabs[m + 1], ctx->sym, &tot);
        void *p = ctx->be->alloc(sizeof(double) * tot);
        out.push_back(p);
        if (on_device) ctx->be->copy(p, iso[m], sizeof(double) * tot);
        else ctx->be->upload(p, iso[m], sizeof(double) * tot);
      }
    };
    take(ctx->ltab, left_iso, nl, ctx->liso);
    take(ctx->rtab, right_iso, nr, ctx->riso);
    ctx->be->sync();
  }
  ctx->have_mps = true;
  GUARD_END
}

int dmrg_build_env(dmrg_ctx *ctx, int precision, int slices) {
  GUARD_BEGIN
  need_gpu(ctx);
  const int kappa = check_precision(precision, slices);
  if (!ctx->have_mps) throw StateError("dmrg_build_env before dmrg_set_mps");
  ctx->drop_env();
  ctx->left = vacuum_block(ctx, ctx->ltab[0]);
  for (int m = 0; m < ctx->bond; ++m) renorm_step(ctx, ctx->left, m, true, ctx->ltab[m + 1], ctx->liso[m], false, kappa);
  ctx->right = vacuum_block(ctx, ctx->rtab[0]);
  int nr = ctx->L - ctx->bond - 2;
  for (int m = 0; m < nr; ++m)
    renorm_step(ctx, ctx->right, ctx->L - 1 - m, false, ctx->rtab[m + 1], ctx->riso[m], false, kappa);
  ctx->env_ready = true;
  prepare_heff(ctx, kappa);
  GUARD_END
}

int dmrg_plan_bond(dmrg_ctx *ctx) {
  GUARD_BEGIN
  if (!ctx->have_mps) throw StateError("dmrg_plan_bond before dmrg_set_mps");
  if (ctx->be) throw StateError("dmrg_plan_bond is for planning contexts; use dmrg_build_env");
  ctx->drop_env();
  auto lay = [&](BlockState &b, const BondTable &tab, int first, int n) {
    b = BlockState();
    b.sym = ctx->sym;
    b.tab = tab; b.n_orb = n;
    for (int p = first; p < first + n; ++p) {
      if (ctx->sym == DMRG_SYM_U1U1) { b.orbs.push_back(2 * p); b.orbs.push_back(2 * p + 1); } else b.orbs.push_back(p);
    }
    layout_block(b, ctx->L);
  };
  lay(ctx->left, ctx->ltab.back(), 0, ctx->bond);
  lay(ctx->right, ctx->rtab.back(), ctx->bond + 2, ctx->L - ctx->bond - 2);
  ctx->env_ready = true;
  prepare_heff(ctx);
  GUARD_END
}

int dmrg_split_truncate(dmrg_ctx *ctx, const double *psi, int on_device, int direction, int64_t max_states,
                        double *discarded) {
  GUARD_BEGIN
  if (!ctx->plan_ready) throw StateError("dmrg_split_truncate before dmrg_build_env / dmrg_plan_bond");
  if (!psi || max_states < 1) throw std::invalid_argument("dmrg_split_truncate: bad arguments");
  if (direction != DMRG_LEFT_TO_RIGHT && direction != DMRG_RIGHT_TO_LEFT) throw std::invalid_argument("bad direction");
  std::vector<double> host;
  if (on_device) {
    need_gpu(ctx);
    host.resize((size_t)ctx->plan.psi_len);
    ctx->be->download(host.data(), psi, sizeof(double) * host.size());
    psi = host.data();
  }
  const bool l2r = direction == DMRG_LEFT_TO_RIGHT;
  split_truncate(ctx->plan, l2r ? ctx->left.tab : ctx->right.tab, ctx->sym, l2r, psi, max_states, ctx->split);
  if (discarded) *discarded = ctx->split.discarded;
  GUARD_END
}

int dmrg_split_result(dmrg_ctx *ctx, const int64_t **table, int64_t *table_rows, const double **isometry,
                      int64_t *isometry_len) {
  GUARD_BEGIN
  if (!table || !table_rows || !isometry || !isometry_len) throw std::invalid_argument("null output");
  if (ctx->split.table.empty()) throw StateError("dmrg_split_result before dmrg_split_truncate");
  *table = ctx->split.table.data(); *table_rows = (int64_t)ctx->split.table.size() / 4;
  *isometry = ctx->split.iso.data(); *isometry_len = (int64_t)ctx->split.iso.size();
  GUARD_END
}

int dmrg_replan(dmrg_ctx *ctx, int precision, int slices) {
  GUARD_BEGIN
  const int kappa = check_precision(precision, slices);
  if (!ctx->plan_ready) throw StateError("dmrg_replan before dmrg_build_env / dmrg_plan_bond");
  ensure_plan(ctx, kappa);
  GUARD_END
}

int dmrg_psi_length(dmrg_ctx *ctx, int64_t *n) {
  GUARD_BEGIN
  if (!ctx->plan_ready) throw StateError("no H_eff plan: call dmrg_build_env (or dmrg_plan_bond) first");
  if (!n) throw std::invalid_argument("null output");
  *n = ctx->plan.psi_len;
  GUARD_END
}

int dmrg_heff_apply(dmrg_ctx *ctx, const double *psi_in_dev, double *psi_out_dev, int precision, int slices) {
  GUARD_BEGIN
  need_gpu(ctx);
  const int kappa = check_precision(precision, slices);
  ctx->performant = precision == DMRG_PREC_FP64_EMU_PERF;
  if (!ctx->plan_ready) throw StateError("dmrg_heff_apply before dmrg_build_env");
  if (!psi_in_dev || !psi_out_dev || psi_in_dev == psi_out_dev) throw std::invalid_argument("dmrg_heff_apply: bad pointers");
  ensure_plan(ctx, kappa);
  heff_apply(ctx, psi_in_dev, psi_out_dev);
  GUARD_END
}

int dmrg_heff_apply_host(dmrg_ctx *ctx, const double *psi_in_host, double *psi_out_host, int precision, int slices) {
  GUARD_BEGIN
  need_gpu(ctx);
  const int kappa = check_precision(precision, slices);
  ctx->performant = precision == DMRG_PREC_FP64_EMU_PERF;
  if (!ctx->plan_ready) throw StateError("dmrg_heff_apply_host before dmrg_build_env");
  if (!psi_in_host || !psi_out_host) throw std::invalid_argument("dmrg_heff_apply_host: bad pointers");
  ensure_plan(ctx, kappa);
  size_t bytes = sizeof(double) * ctx->plan.psi_len;
  if (!ctx->psi_a) { ctx->psi_a = ctx->be->alloc(bytes); ctx->psi_b = ctx->be->alloc(bytes); }
  ctx->be->upload(ctx->psi_a, psi_in_host, bytes);
  heff_apply(ctx, (const double *)ctx->psi_a, (double *)ctx->psi_b);
  ctx->be->download(psi_out_host, ctx->psi_b, bytes);
  GUARD_END
}

int dmrg_heff_diag(dmrg_ctx *ctx, double *diag_out_dev) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!ctx->plan_ready) throw StateError("dmrg_heff_diag before dmrg_build_env");
  if (!diag_out_dev) throw std::invalid_argument("null output");
  BufTable bt = heff_bufs(ctx, nullptr, nullptr);
  ctx->be->run_diag(ctx->d_diag, bt, diag_out_dev);
  GUARD_END
}

// Two-site sweeps on the device.  Every bond: H_eff plan on the stacked
// blocks, restarted Davidson from a seeded random start, split and truncate (a10), one renormalization (a9) that
// pushes the grown block onto its stack.  The blocks of both sides stay resident.
int dmrg_sweep(dmrg_ctx *ctx, int n_sweeps, int64_t max_states, int davidson_iters, int max_restarts, double tol,
               int precision, int slices, uint64_t seed, double *energies, int64_t *n_energies, double *max_discarded) {
  GUARD_BEGIN
  need_gpu(ctx);
  const int kappa = check_precision(precision, slices);
  ctx->performant = precision == DMRG_PREC_FP64_EMU_PERF;
  const int L = ctx->L;
  if (!ctx->have_mps || ctx->bond != 0) throw StateError("dmrg_sweep needs dmrg_set_mps at bond 0 (right-canonical start)");
  if (n_sweeps < 1 || max_states < 1 || davidson_iters < 2 || davidson_iters > MAX_DAVIDSON || max_restarts < 1 ||
      !energies || !n_energies || *n_energies < (int64_t)2 * (L - 1) * n_sweeps)
    throw std::invalid_argument("dmrg_sweep: bad arguments (energies must hold 2 (L - 1) n_sweeps values)");
  Backend &be = *ctx->be;
  ctx->drop_env();
  ctx->drop_stacks();
  // stacks: lstack[m] / rstack[m] = block of m sites; the right stack is built from the start state
  ctx->lstack.push_back(vacuum_block(ctx, ctx->ltab[0]));
  ctx->rstack.push_back(vacuum_block(ctx, ctx->rtab[0]));
  for (int m = 0; m < L - 2; ++m) {
    BlockState nb = ctx->rstack[m];
    renorm_step(ctx, nb, L - 1 - m, false, ctx->rtab[m + 1], ctx->riso[m], true, kappa);
    ctx->rstack.push_back(nb);
  }
  std::vector<BondTable> LT = ctx->ltab, RT = ctx->rtab;       // tables by number of absorbed sites
  std::vector<void *> LI = ctx->liso, RI = ctx->riso;          // device isometries (owned by the context lists)
  LT.resize(L - 1); LI.resize(L - 2, nullptr);
  ctx->lstack.resize(1);
  int64_t n_e = 0;
  double worst = 0.0;
  uint64_t rng = seed * 0x9E3779B97F4A7C15ull + 0xD1B54A32D192ED03ull;
  auto next_uniform = [&]() {                                   // splitmix64 -> (-1, 1)
    rng += 0x9E3779B97F4A7C15ull;
    uint64_t z = rng;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull; z = (z ^ (z >> 27)) * 0x94D049BB133111EBull; z ^= z >> 31;
    return (double)(z >> 11) * (2.0 / 9007199254740992.0) - 1.0;
  };
  std::vector<double> host, th(davidson_iters), rs(davidson_iters);
  void *psi_dev = nullptr;
  int64_t psi_cap = 0;
  auto solve = [&](int p) {
    const int nl = p, nr = L - p - 2;
    ctx->drop_plan();
    ctx->left = ctx->lstack[nl]; ctx->right = ctx->rstack[nr];
    ctx->env_borrowed = true; ctx->env_ready = true; ctx->bond = p;
    ctx->ltab.assign(LT.begin(), LT.begin() + nl + 1);          // the tables of this bond (dmrg_table, plan)
    ctx->rtab.assign(RT.begin(), RT.begin() + nr + 1);
    prepare_heff(ctx, kappa);
    const int64_t n = ctx->plan.psi_len;
    if (n > psi_cap) { be.release(psi_dev); psi_dev = nullptr; psi_dev = be.alloc(sizeof(double) * n); psi_cap = n; }
    host.resize((size_t)n);
    for (auto &x : host) x = next_uniform();
    be.upload(psi_dev, host.data(), sizeof(double) * n);
    const int it = (int)std::min<int64_t>(davidson_iters, n);
    double e = 0.0;
    for (int r = 0; r < max_restarts; ++r) {
      const int done = davidson_run(ctx, (double *)psi_dev, it, tol, th.data(), rs.data());
      e = th[done - 1];
      if (rs[done - 1] < tol) break;
    }
    energies[n_e++] = e + ctx->ints.e_core;
  };
  auto grow = [&](int p, bool l2r) {
    double disc = 0.0;
    host.resize((size_t)ctx->plan.psi_len);
    be.download(host.data(), psi_dev, sizeof(double) * host.size());
    split_truncate(ctx->plan, l2r ? ctx->left.tab : ctx->right.tab, ctx->sym, l2r, host.data(), max_states, ctx->split);
    disc = ctx->split.discarded;
    worst = std::max(worst, disc);
    const BondTable nt = make_table(ctx->split.table.data(), (int64_t)ctx->split.table.size() / 4);
    void *iso = be.alloc(sizeof(double) * std::max<size_t>(ctx->split.iso.size(), 1));
    be.upload(iso, ctx->split.iso.data(), sizeof(double) * ctx->split.iso.size());
    be.sync();
    const int m = l2r ? p : L - p - 2;                          // sites in the block that grows
    std::vector<BlockState> &stack = l2r ? ctx->lstack : ctx->rstack;
    std::vector<BondTable> &T = l2r ? LT : RT;
    std::vector<void *> &I = l2r ? LI : RI;
    for (size_t k = m + 1; k < stack.size(); ++k) be.release(stack[k].dev);   // blocks built on the old isometry
    stack.resize(m + 1);
    BlockState nb = stack[m];
    renorm_step(ctx, nb, l2r ? p : p + 1, l2r, nt, iso, true, kappa);
    stack.push_back(nb);
    T[m + 1] = nt;
    be.release(I[m]); I[m] = iso;
  };
  try {
    // "the sweeping procedure was terminated once the energy difference between three subsequent sweeps
    // dropped below eps_sweep" -- option sweep_eps (0 = run all n_sweeps); the energy of a sweep is its lowest bond energy
    std::vector<double> e_sweep;
    for (int sw = 0; sw < n_sweeps; ++sw) {
      const int64_t first = n_e;
      for (int p = 0; p <= L - 2; ++p) { solve(p); if (p < L - 2) grow(p, true); }
      for (int p = L - 2; p >= 0; --p) { solve(p); if (p > 0) grow(p, false); }
      e_sweep.push_back(*std::min_element(energies + first, energies + n_e));
      const size_t n = e_sweep.size();
      if (ctx->opt.sweep_eps > 0 && n >= 3 && std::fabs(e_sweep[n - 1] - e_sweep[n - 2]) < ctx->opt.sweep_eps &&
          std::fabs(e_sweep[n - 2] - e_sweep[n - 3]) < ctx->opt.sweep_eps)
        break;
    }
  } catch (...) {        // leave a consistent, empty context: the caller starts again from dmrg_set_mps
    be.release(psi_dev);
    ctx->liso.clear(); ctx->riso.clear();            // LI / RI hold every live isometry (replaced ones were released)
    for (void *q : LI) if (q) ctx->liso.push_back(q);
    for (void *q : RI) if (q) ctx->riso.push_back(q);
    ctx->drop_plan();
    ctx->drop_stacks();
    ctx->drop_mps();
    throw;
  }
  be.release(psi_dev);
  // leave the context with the final right-canonical state at bond 0 (left = vacuum) and no environments
  for (void *q : LI) be.release(q);
  ctx->liso.clear(); ctx->riso = RI;
  LT.resize(1);
  ctx->ltab = LT; ctx->rtab = RT;
  ctx->drop_plan();
  ctx->drop_stacks();
  *n_energies = n_e;
  if (max_discarded) *max_discarded = worst;
  GUARD_END
}

int dmrg_davidson_step(dmrg_ctx *ctx, double *psi, int n_iter, double tol, int precision, int slices,
                       double *theta_host, double *resid_host, int *n_done) {
  GUARD_BEGIN
  need_gpu(ctx);
  const int kappa = check_precision(precision, slices);
  ctx->performant = precision == DMRG_PREC_FP64_EMU_PERF;
  if (!ctx->plan_ready) throw StateError("dmrg_davidson_step before dmrg_build_env");
  if (!psi || n_iter < 1 || n_iter > MAX_DAVIDSON || !theta_host || !resid_host || !n_done)
    throw std::invalid_argument("dmrg_davidson_step: bad arguments (1 <= n_iter <= 32)");
  ensure_plan(ctx, kappa);
  *n_done = davidson_run(ctx, psi, n_iter, tol, theta_host, resid_host);
  GUARD_END
}

int dmrg_renormalize(dmrg_ctx *ctx, int direction, const int64_t *new_table, int64_t new_rows, const double *isometry,
                     int on_device, int precision, int slices) {
  GUARD_BEGIN
  need_gpu(ctx);
  const int kappa = check_precision(precision, slices);
  if (!ctx->env_ready) throw StateError("dmrg_renormalize before dmrg_build_env");
  if (ctx->env_borrowed) throw StateError("dmrg_renormalize while a sweep owns the blocks");
  if (!new_table || new_rows < 1 || !isometry) throw std::invalid_argument("dmrg_renormalize: bad arguments");
  if (direction != DMRG_LEFT_TO_RIGHT && direction != DMRG_RIGHT_TO_LEFT) throw std::invalid_argument("bad direction");
  BondTable nt = make_table(new_table, new_rows);
  bool l2r = direction == DMRG_LEFT_TO_RIGHT;
  BlockState &blk = l2r ? ctx->left : ctx->right;
  int site = l2r ? ctx->bond : ctx->bond + 1;
  int64_t tot = 0;
  iso_blocks(blk.tab, nt, ctx->sym, &tot);
  ctx->drop_plan();
  void *iso = ctx->be->alloc(sizeof(double) * tot);
  try {
    if (on_device) ctx->be->copy(iso, isometry, sizeof(double) * tot);
    else ctx->be->upload(iso, isometry, sizeof(double) * tot);
    renorm_step(ctx, blk, site, l2r, nt, iso, false, kappa);
  } catch (...) { ctx->be->release(iso); throw; }
  ctx->be->release(iso);
  ctx->tab_bondL = table_rows(ctx->left.tab);
  ctx->tab_bondR = table_rows(ctx->right.tab);
  GUARD_END
}

int dmrg_table(dmrg_ctx *ctx, int which, const int64_t **data, int64_t *count) {
  GUARD_BEGIN
  if (!data || !count) throw std::invalid_argument("null output");
  const std::vector<int64_t> *v = nullptr;
  if (which == DMRG_TAB_BOND_L || which == DMRG_TAB_BOND_R) {
    if (!ctx->env_ready) throw StateError("no environment");
    v = which == DMRG_TAB_BOND_L ? &ctx->tab_bondL : &ctx->tab_bondR;
  } else {
    if (!ctx->plan_ready) throw StateError("no H_eff plan: call dmrg_build_env (or dmrg_plan_bond) first");
    switch (which) {
      case DMRG_TAB_PSI_BLOCKS: v = &ctx->plan.tab_psi; break;
      case DMRG_TAB_OP_BLOCKS_L: v = &ctx->plan.tab_opL; break;
      case DMRG_TAB_OP_BLOCKS_R: v = &ctx->plan.tab_opR; break;
      case DMRG_TAB_GROUPS: v = &ctx->plan.tab_groups; break;
      case DMRG_TAB_FALG: v = &ctx->tab_falg; break;
      case DMRG_TAB_COUNTS: v = &ctx->plan.tab_counts; break;
      case DMRG_TAB_ISO_BLOCKS_L: v = &ctx->tab_isoL; break;
      case DMRG_TAB_ISO_BLOCKS_R: v = &ctx->tab_isoR; break;
      case DMRG_TAB_FALG_BLOCKS: v = &ctx->plan.tab_falg_blocks; break;
      default: throw std::invalid_argument("unknown table id");
    }
  }
  *data = v->data();
  *count = (int64_t)v->size();
  GUARD_END
}

int dmrg_op_export(dmrg_ctx *ctx, int side, int kind, int i, int k, double *dense, int64_t dim) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!ctx->env_ready) throw StateError("dmrg_op_export before dmrg_build_env");
  if (!dense || (side != 0 && side != 1)) throw std::invalid_argument("dmrg_op_export: bad arguments");
  const BlockState &b = side == 0 ? ctx->left : ctx->right;
  if (dim != b.tab.total) throw std::invalid_argument("dmrg_op_export: dim must equal the block dimension");
  const int rank = kind >> 8;          // SU(2): doubled rank of A / B in bits 8.. (0 or 2)
  kind &= 0xff;
  if (kind < DMRG_OP_I || kind > DMRG_OP_B) throw std::invalid_argument("unknown operator kind");
  Sym s{kind, 0, i, k};
  if (b.sym != 0 && (kind == K_A || kind == K_B)) s.rank = rank;
  if (kind == K_I || kind == K_H) { s.i = s.k = -1; }
  if (kind == K_C || kind == K_S) s.k = -1;
  int cls = b.find_class(kind, sym_class(s, b.sym));
  if (cls < 0) throw std::invalid_argument("operator not stored by this block");
  const OpClass &oc = b.classes[cls];
  auto it = oc.member_index.find({s.i, s.k});
  if (it == oc.member_index.end()) throw std::invalid_argument("operator not stored by this block");
  std::fill(dense, dense + dim * dim, 0.0);
  std::vector<double> tmp;
  for (const OpBlock &ob : oc.blocks) {
    const Sector &qb = b.tab.sec[ob.bra], &qk = b.tab.sec[ob.ket];
    int64_t e = qb.dim * qk.dim;
    tmp.resize(e);
    ctx->be->download(tmp.data(), (const double *)b.dev + ob.off + (int64_t)it->second * e, sizeof(double) * e);
    for (int64_t r = 0; r < qb.dim; ++r)
      for (int64_t c = 0; c < qk.dim; ++c) dense[(qb.off + r) * dim + qk.off + c] = tmp[r * qk.dim + c];
  }
  GUARD_END
}

int dmrg_op_export_class(dmrg_ctx *ctx, int side, int kind, int i0, int k0, int i_bra, int i_ket, double *out,
                         int64_t capacity, int64_t *members, int64_t member_capacity, int64_t *n_members,
                         int64_t *rows, int64_t *cols) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!ctx->env_ready) throw StateError("dmrg_op_export_class before dmrg_build_env");
  if (!n_members || !rows || !cols || (side != 0 && side != 1)) throw std::invalid_argument("dmrg_op_export_class: bad arguments");
  const BlockState &b = side == 0 ? ctx->left : ctx->right;
  const int rank = kind >> 8;
  kind &= 0xff;
  if (kind < DMRG_OP_I || kind > DMRG_OP_B) throw std::invalid_argument("unknown operator kind");
  const int ns = (int)b.tab.sec.size();
  if (i_bra < 0 || i_bra >= ns || i_ket < 0 || i_ket >= ns) throw std::invalid_argument("sector index out of range");
  Sym s{kind, 0, i0, k0};
  if (b.sym != 0 && (kind == K_A || kind == K_B)) s.rank = rank;
  *n_members = 0; *rows = b.tab.sec[i_bra].dim; *cols = b.tab.sec[i_ket].dim;
  const int cls = b.find_class(kind, sym_class(s, b.sym));
  if (cls < 0) return DMRG_OK;
  const OpClass &oc = b.classes[cls];
  auto it = oc.block_index.find({i_bra, i_ket});
  if (it == oc.block_index.end()) return DMRG_OK;
  *n_members = oc.n();
  if (!out) return DMRG_OK;
  const int64_t e = *rows * *cols * oc.n();
  if (capacity < e || !members || member_capacity < oc.n()) throw std::invalid_argument("dmrg_op_export_class: buffers too small");
  for (int a = 0; a < oc.n(); ++a) { members[2 * a] = oc.members[a].first; members[2 * a + 1] = oc.members[a].second; }
  ctx->be->download(out, (const double *)b.dev + oc.blocks[it->second].off, sizeof(double) * e);
  GUARD_END
}

int dmrg_set_timing(dmrg_ctx *ctx, int enable) {
  GUARD_BEGIN
  ctx->timing = enable != 0;
  GUARD_END
}

int dmrg_last_emu_ms(dmrg_ctx *ctx, double *ms_slice, double *ms_int8) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!ctx->timing) throw StateError("timing is disabled (dmrg_set_timing)");
  if (!ms_slice || !ms_int8) throw std::invalid_argument("null output");
  *ms_slice = ctx->ms_slice;
  *ms_int8 = ctx->ms_int8;
  GUARD_END
}

int dmrg_last_emu_stage1_ms(dmrg_ctx *ctx, double *ms_tensor) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!ctx->timing) throw StateError("timing is disabled (dmrg_set_timing)");
  if (!ms_tensor) throw std::invalid_argument("null output");
  *ms_tensor = ctx->ms_s1_tensor;
  GUARD_END
}

int dmrg_last_stage_ms(dmrg_ctx *ctx, double *ms1, double *ms2) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!ctx->timing) throw StateError("timing is disabled (dmrg_set_timing)");
  if (!ms1 || !ms2) throw std::invalid_argument("null output");
  *ms1 = ctx->ms1;
  *ms2 = ctx->ms2;
  GUARD_END
}

int dmrg_emu_gemm(dmrg_ctx *ctx, int M, int N, int K, const double *A, const double *B, double *C, int slices,
                  double *ms_slice, double *ms_gemm) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!A || !B || !C) throw std::invalid_argument("dmrg_emu_gemm: null pointer");
  ctx->be->emu_gemm(M, N, K, A, B, C, slices == 0 ? 6 : slices, slices == 0 ? 6 : slices, ms_slice, ms_gemm);
  GUARD_END
}

int dmrg_emu_gemm_kept(dmrg_ctx *ctx, int M, int N, int K, const double *A, const double *B, double *C, int slices, int keep) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!A || !B || !C) throw std::invalid_argument("dmrg_emu_gemm_kept: null pointer");
  ctx->be->emu_gemm(M, N, K, A, B, C, slices == 0 ? 6 : slices, keep, nullptr, nullptr);
  GUARD_END
}

int dmrg_emu_sum_perf(dmrg_ctx *ctx, int M, int N, int K, int n, const double *A, const double *B, const double *alpha_host,
                      double *C, int slices, int kmin, int32_t *keep_out_host) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!A || !B || !C || !alpha_host || !keep_out_host) throw std::invalid_argument("dmrg_emu_sum_perf: null pointer");
  if (kmin < 1 || kmin > 7) throw std::invalid_argument("dmrg_emu_sum_perf: kmin in [1, 7]");
  std::vector<int> keep(std::max(n, 0));
  ctx->be->emu_sum(M, N, K, n, A, B, alpha_host, C, slices == 0 ? 6 : slices, kmin, keep.data());
  for (int g = 0; g < n; ++g) keep_out_host[g] = keep[g];
  GUARD_END
}

int dmrg_emu_keep_rule(dmrg_ctx *ctx, const int32_t *E_all, const int32_t *E_nz, int n, int slices, int kmin, int32_t *keep_out) {
  GUARD_BEGIN
  if (n < 0 || (n > 0 && (!E_all || !E_nz || !keep_out))) throw std::invalid_argument("dmrg_emu_keep_rule: bad arguments");
  const int kappa = slices == 0 ? 6 : slices;
  if (kappa < 2 || kappa > 7 || kmin < 1 || kmin > 7) throw std::invalid_argument("dmrg_emu_keep_rule: slices in [2, 7], kmin in [1, 7]");
  int ref = EMU_NO_REF;
  for (int i = 0; i < n; ++i) if (E_nz[i] != DMRG_EMU_NO_REF) ref = std::max(ref, (int)E_nz[i]);
  for (int i = 0; i < n; ++i) keep_out[i] = ref == EMU_NO_REF ? kappa : emu_keep_rule(kappa, kmin, ref, E_all[i]);
  GUARD_END
}

int dmrg_launch_count(dmrg_ctx *ctx, uint64_t *n) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!n) throw std::invalid_argument("dmrg_launch_count: null pointer");
  *n = ctx->be->launch_count();
  GUARD_END
}

int dmrg_last_emu_products(dmrg_ctx *ctx, uint64_t *kept, uint64_t *eager) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!kept || !eager) throw std::invalid_argument("dmrg_last_emu_products: null pointer");
  uint64_t v[2] = {0, 0};
  if (ctx->plan_ready && ctx->emu_kappa >= 2 && ctx->emu_kappa <= 7) ctx->be->emu_products(ctx->d_emu, v);
  *kept = v[0]; *eager = v[1];
  GUARD_END
}

int dmrg_tf32_split(dmrg_ctx *ctx, const double *src_dev, int64_t n, uint32_t *hi_dev, uint32_t *lo_dev) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (n < 0 || (n > 0 && (!src_dev || !hi_dev || !lo_dev))) throw std::invalid_argument("dmrg_tf32_split: bad arguments");
  ctx->be->tf32_split_run(src_dev, n, hi_dev, lo_dev);
  ctx->be->sync();
  GUARD_END
}

int dmrg_emu_slice(dmrg_ctx *ctx, const double *src, int lines, int K, int64_t line_stride, int64_t k_stride,
                   int slices, signed char *out, int *expo) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!src || !out || !expo || lines < 1 || K < 1) throw std::invalid_argument("dmrg_emu_slice: bad arguments");
  ctx->be->emu_slice(src, lines, K, line_stride, k_stride, slices == 0 ? 6 : slices, out, expo);
  ctx->be->sync();
  GUARD_END
}

int dmrg_dots(dmrg_ctx *ctx, const double *V, int64_t ld, int nvec, const double *w, int64_t n, double *out) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!V || !w || !out || nvec < 1 || nvec > MAX_DAVIDSON || n < 0 || ld < 0)
    throw std::invalid_argument("dmrg_dots: bad arguments (1 <= nvec <= 32)");
  ctx->be->dots(V, ld, nvec, w, n, out);
  GUARD_END
}

// HBM-class kernels of the path, each timed alone with CUDA events on the context's stream ("achieved
// HBM GB/s" for the kernels that are bound by bandwidth, not by a tensor pipe).  bytes = ALGORITHMIC bytes of one launch.
int dmrg_measure_hbm_kernels(dmrg_ctx *ctx, const double *psi_dev, int n_basis, double *ms_out, double *bytes_out,
                             int capacity, int *n_out) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!ctx->plan_ready) throw StateError("dmrg_measure_hbm_kernels before dmrg_build_env");
  if (!psi_dev || !ms_out || !bytes_out || !n_out || capacity < DMRG_HBM_N || n_basis < 1 || n_basis > MAX_DAVIDSON)
    throw std::invalid_argument("dmrg_measure_hbm_kernels: bad arguments");
  Backend &be = *ctx->be;
  const HeffPlan &P = ctx->plan;
  const int64_t n = P.psi_len;
  const int m = n_basis, reps = 5;
  for (int i = 0; i < DMRG_HBM_N; ++i) { ms_out[i] = 0.0; bytes_out[i] = 0.0; }
  void *tmp = be.alloc(sizeof(double) * ((2 * (int64_t)m + 4) * n + 64));
  try {
    double *V = (double *)tmp, *W = V + (int64_t)m * n, *x = W + (int64_t)m * n, *r = x + n, *t = r + n, *dg = t + n,
           *sc = dg + n;
    for (int v = 0; v < m; ++v) { be.copy(V + (int64_t)v * n, psi_dev, sizeof(double) * n); be.copy(W + (int64_t)v * n, psi_dev, sizeof(double) * n); }
    be.zero(sc, sizeof(double) * 64);
    BufTable bt = heff_bufs(ctx, psi_dev, t);
    auto timed = [&](int slot, double bytes, const std::function<void()> &launch) {
      launch();                                            // warm-up
      be.timer_mark(4);
      for (int i = 0; i < reps; ++i) launch();
      be.timer_mark(5);
      ms_out[slot] = be.timer_ms(4, 5) / reps;
      bytes_out[slot] = bytes;
    };
    double diag_reads = 0;
    for (const DiagJob &j : P.diag_jobs) diag_reads += 8.0 * (j.t_end - j.t_begin) * (j.dL + j.dR);
    timed(DMRG_HBM_DIAG, 8.0 * n + diag_reads, [&] { be.run_diag(ctx->d_diag, bt, dg); });
    timed(DMRG_HBM_DOTS, 8.0 * n * (m + 1), [&] { be.dots(V, n, m, W, n, sc); });
    be.dots(V, n, 1, V, n, sc + 40);                       // a finite theta for the kernels below
    timed(DMRG_HBM_RITZ, 8.0 * n * (2 * m + 2), [&] { be.ritz_residual(V, W, n, m, n, sc, sc + 40, x, r); });
    timed(DMRG_HBM_PRECOND, 8.0 * n * 3, [&] { be.precondition(r, dg, sc + 40, t, n); });
    timed(DMRG_HBM_PROJECT, 8.0 * n * (m + 2), [&] { be.subtract_projection(V, n, m, sc, t, n); });
    if (ctx->emu_kappa) {
      const double bpe = ctx->emu_kappa;                   // bytes per sliced element: kappa INT8 digits, or 8 (hi + lo TF32)
      auto elems = [](const std::vector<EmuSliceDesc> &v, bool skip_fused) {
        double e = 0;
        for (const EmuSliceDesc &d : v) if (!(skip_fused && d.bound == 2)) e += (double)d.lines * d.n_members * d.dl;
        return e;
      };
      const double ep = elems(P.sliceP, false), el = elems(P.sliceL, false), er = elems(P.sliceR, false);
      if (ep > 0) timed(DMRG_HBM_SLICE_PSI, (8.0 + bpe) * ep, [&] { be.run_emu_slice(ctx->d_emu, EMU_SLICE_PSI, bt); });
      if (el > 0) timed(DMRG_HBM_SLICE_OPS_L, (8.0 + bpe) * el, [&] { be.run_emu_slice(ctx->d_emu, EMU_SLICE_L, bt); });
      if (er > 0) timed(DMRG_HBM_SLICE_OPS_R, (8.0 + bpe) * er, [&] { be.run_emu_slice(ctx->d_emu, EMU_SLICE_R, bt); });
      // T of pass 0 (the part that is not emitted by the stage-1 epilogue): needs the T of a stage-1 run in the scratch
      const double et = P.emu.empty() ? 0.0 : elems(P.emu[0].sliceT, true);
      if (et > 0) {
        be.run_emu_norms(ctx->d_emu, 0, bt);
        be.run_jobs(ctx->d_stage1[0], bt);
        timed(DMRG_HBM_SLICE_T, (8.0 + bpe) * et, [&] { be.run_emu_slice(ctx->d_emu, 0, bt); });
      }
    }
    be.sync();
  } catch (...) { be.release(tmp); throw; }
  be.release(tmp);
  *n_out = DMRG_HBM_N;
  GUARD_END
}

int dmrg_measure_peak(dmrg_ctx *ctx, int which, double *ops_per_s) {
  GUARD_BEGIN
  need_gpu(ctx);
  if (!ops_per_s) throw std::invalid_argument("null output");
  *ops_per_s = ctx->be->measure_peak(which);
  GUARD_END
}

}  // extern "C"
