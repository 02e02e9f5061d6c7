/* dmrg.h -- C ABI of the B200-native two-site DMRG hot path.
 *
 * What the library computes (citations: PAPER.md = /root/reference/PAPER.md of
 * arxiv/paper_2603_28648; SURVEY.md / DESIGN.md in this repository):
 *   - the two-site effective-Hamiltonian product H_eff.psi applied inside each
 *     eigen-solver step of DMRG ("Method", "Numerical procedure";
 *     SURVEY.md section 8(a) rows a5, a6, Appendix A5),
 *   - the renormalization step that builds the next block's operators
 *     (the O(N^2 D^2) operator set),
 *   - the Davidson vector work on device ("Lanczos", residual 1e-6;
 *     DESIGN.md reading s6).
 * The problem statement is the ab initio Hamiltonian in the site basis
 * {|0>,|u>,|d>,|ud>} of PAPER.md:41 with one-electron integrals h_ij and
 * two-electron integrals V_ijkl = (ij|kl) (chemists' order), N electrons, 2S (or
 * 2S_z) and a block-state budget D (BASELINE.json north_star).
 *
 * Conventions for every call:
 *   - returns DMRG_OK (0) or a negative error code; no exception or abort crosses
 *     the ABI; dmrg_last_error() gives a borrowed message for the last failure;
 *   - "host" pointers are read during the call and copied; "device" pointers are
 *     caller-owned CUDA device memory that must outlive the stream work using it;
 *     the library never frees or reallocates caller memory;
 *   - all device work is enqueued on the context's stream; only calls that return
 *     host scalars (documented below) synchronise;
 *   - there is no CPU fallback: compute calls on a context without a usable
 *     sm_100 device fail with DMRG_EUNSUPPORTED.  A context created with
 *     device < 0 is a PLANNING context: it builds the integer tables only
 *     (dmrg_table works after dmrg_plan_bond) and every compute call fails.
 *
 * Packed layouts:
 *   bond table rows   (N, twoS, dim, offset) int64, sorted by (N, twoS); twoS is
 *                     2S_z for DMRG_SYM_U1U1;
 *   isometry blocks   (i_prev, s, i_next) lexicographic, each row-major
 *                     [a_prev][a_next], blocks contiguous;
 *   psi blocks        (iL, s1, s2, iR) lexicographic, each row-major [l][r];
 *   site state index  0=|0>, 1=|u>, 2=|d>, 3=|ud> = a+_u a+_d |0>.
 */
#ifndef DMRG_B200_H
#define DMRG_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dmrg_ctx dmrg_ctx;

enum { DMRG_OK = 0, DMRG_EINVAL = -1, DMRG_ESTATE = -2, DMRG_ENOMEM = -3,
       DMRG_ECUDA = -4, DMRG_EUNSUPPORTED = -5 };
enum { DMRG_SYM_U1U1 = 0, DMRG_SYM_SU2 = 1 };
/* precision modes: native FP64 (DMMA), Ozaki-emulated FP64 on INT8 tensor cores
 * (kappa = 6 slices), 3xTF32 (hi/lo TF32 split, three products, FP32 accumulation;
 * DESIGN.md reading s15, tolerance 1e-5; `slices` is ignored).  In the two tensor-core modes the stage-1 jobs
 * and two-sided stage-2 segments above a size threshold run on tcgen05, the rest stays native FP64; the
 * renormalization runs its two rotation products in the mode it is called with; the contracted-operator build (a3)
 * is native FP64 in every mode. */
enum { DMRG_PREC_FP64 = 0, DMRG_PREC_FP64_EMU = 1, DMRG_PREC_TF32X3 = 2,
       /* PAPER.md:53, 59 "performant mode ... dynamic mantissa bit settings" (DESIGN.md reading
        * s21): emulated FP64 with `slices` = kappa as in DMRG_PREC_FP64_EMU (the paper's "eager mode"), but every task
        * class (one stage-2 segment: an operator-pair class meeting one psi block) forms only the slice products
        * s + t <= keep + 1, keep = kappa - floor((E_ref - E_class) / 8) >= option emu_kmin (default 3), from the exponents
        * of the class magnitudes inside its output block -- decided on the device at every apply.  Accepted by
        * dmrg_heff_apply(_host), dmrg_davidson_step, dmrg_sweep; dmrg_renormalize / dmrg_build_env treat it as
        * DMRG_PREC_FP64_EMU. */
       DMRG_PREC_FP64_EMU_PERF = 3 };
enum { DMRG_LEFT_TO_RIGHT = 0, DMRG_RIGHT_TO_LEFT = 1 };
/* dmrg_table ids.  All tables are int64. */
enum {
  DMRG_TAB_BOND_L = 0,     /* rows (N, twoS, dim, offset) of the left block            */
  DMRG_TAB_BOND_R = 1,     /* same for the right block (its own labels)               */
  DMRG_TAB_PSI_BLOCKS = 2, /* U1U1 rows (iL, s1, s2, iR, dL, dR, offset);
                              SU2 rows (iL, s1, 2S_A, s2, iR, 2S_B, dL, dR, offset)   */
  DMRG_TAB_OP_BLOCKS_L = 3,/* rows (kind, dN, d2S, n_members, i_bra, i_ket, offset)    */
  DMRG_TAB_OP_BLOCKS_R = 4,
  DMRG_TAB_GROUPS = 5,     /* rows (s1', s1, s2', s2, kindL, dagL, kindR, dagR, n)     */
  DMRG_TAB_FALG = 6,       /* one int64: algorithmic flops of one H_eff.psi (8(d))     */
  DMRG_TAB_COUNTS = 7,     /* (n_jobs1, n_segs1, n_jobs2, n_segs2, n_tiles1, n_tiles2,
                              scratch_elems, op_elems_L, op_elems_R, derived_L, derived_R,
                              stage1_flops, stage2_flops, partial_elems, n_passes,
                              emulated_flops, emu_segments, emu_tiles, emulated_stage1_flops): the last four are zero
                              for a native FP64 plan; emulated_flops is the part of stage2_flops
                              that runs on the INT8 tensor cores, emulated_stage1_flops
                              the part of stage1_flops */
  DMRG_TAB_ISO_BLOCKS_L = 8,/* rows (i_prev, s, i_next, rows, cols, offset), last left iso */
  DMRG_TAB_ISO_BLOCKS_R = 9,
  DMRG_TAB_FALG_BLOCKS = 10 /* per psi OUTPUT block: algorithmic flops feeding it (sums to FALG) */
};
/* operator kinds for dmrg_op_export (spin-orbital i = 2*p + sigma, sigma 0 = up):
 * Appendix A2 of SURVEY.md.  I identity, H block Hamiltonian, C_i = a+_i,
 * S_x complement of a+_x, A_ik = a+_i a+_k (i<k), B_il = a+_i a_l.
 * SU(2): spatial orbitals and reduced matrices: C_p = a+_p (rank 1/2),
 * S = S~_x, A^k_pr (p <= r), B^k_ps = [a+_p x a~_s]^k; pass kind | (2k << 8) for A and B. */
enum { DMRG_OP_I = 0, DMRG_OP_H = 1, DMRG_OP_C = 2, DMRG_OP_S = 3, DMRG_OP_A = 4, DMRG_OP_B = 5 };

/* Create a context on CUDA device `device` whose work is enqueued on `cuda_stream`
 * (a cudaStream_t passed as void*; NULL = the legacy default stream).
 * device < 0 creates a planning context (tables only). */
int dmrg_create(dmrg_ctx **out, int device, void *cuda_stream);
int dmrg_destroy(dmrg_ctx *ctx);
/* Plan-time knobs, instead of environment variables (SURVEY.md section 5 "explicit ... parameter on each call; no
 * environment variables").  They select code paths and never change what is computed; the defaults are what bench.py
 * times.  A changed option takes effect when the H_eff plan is next built (the next dmrg_build_env / dmrg_replan /
 * dmrg_heff_apply / dmrg_davidson_step re-plans).  Keys (value is a double; integers must be integral):
 *   emu_mink, emu_minm, emu_minn     stage-2 segment runs on tcgen05 when K, d_L', d_R' reach these (128, 0, 16);
 *                    emu_minm = 0: 8 when the largest sector of the two blocks reaches 96, else 32
 *   emu_mink1, emu_minm1, emu_minn1  stage-1 job runs on tcgen05 when d_R, d_L, n_alpha d_R' reach these (1, 1, 1: all)
 *   emu_stage1 (1)   0: stage 1 stays native FP64 in the tensor-core modes
 *   emu_fuse (1)     0: T is sliced by a separate pass instead of by the stage-1 epilogue
 *   emu_exact_exp (0) 1: exact line maxima for the exponents of T (reading s12b switched off)
 *   emu_gang (1)     0: stage-2 tiles of one job are scheduled independently
 *   emu_s1new (1)    0: emulated stage 1 on the generic segmented kernel instead of k_emu_s1
 *   emu_kmin (3)     DMRG_PREC_FP64_EMU_PERF: fewest slices a task class keeps, in [1, 7]
 *   emu_kpiece (16384) largest K of one emulated stage-2 segment, in [32, 16384]; longer contractions are cut into
 *                    pieces with their own exponents (INT32 accumulators cannot overflow below 16384)
 *   tile (0)         CTA tile edge of the native kernel: 32, 48, 64; 0 = chosen from the sector sizes (the FP64 remainder
 *                    lists of the tensor-core modes: 32)
 *   sweep_eps (0)    dmrg_sweep: stop once the energies of three subsequent sweeps differ by less than this (PAPER.md:51:
 *                    1e-5); 0 = run every sweep asked for.  Does not re-plan.
 *   scratch_gb (0)   budget in GB for the intermediate T of one pass; 0 = default
 *   debug (0)        1: plan statistics on stderr
 * Unknown keys and out-of-range values return DMRG_EINVAL. */
int dmrg_set_option(dmrg_ctx *ctx, const char *key, double value);
const char *dmrg_last_error(dmrg_ctx *ctx);

/* SURVEY.md 8(a) a1.  h: L*L row-major.  V: L^4, V[((i*L+j)*L+k)*L+l] = (ij|kl); may be
 * NULL when chol != NULL (then V = sum_c chol[c][ij] chol[c][kl]).  chol: n_chol*L*L.
 * twoS is 2S for SU2 and 2S_z for U1U1.  D is the block-state budget (informational).
 * Host pointers, copied.  Resets the context to a new problem. */
int dmrg_init_integrals(dmrg_ctx *ctx, int L, const double *h, const double *V,
                        const double *chol, int n_chol, double e_core,
                        int N, int twoS, int symmetry, int D);

/* The state whose environments are built (SURVEY.md Appendix C "Random mixed-canonical
 * MPS").  bond = number of orbitals in the left block; the two-site window is sites
 * (bond, bond+1).  left_tables[m], m = 0..bond: table of the left block with m orbitals;
 * left_iso[m], m = 0..bond-1: packed isometry (table m, site m) -> table m+1.
 * right_tables[m], m = 0..L-bond-2: right block with m orbitals (its own labels);
 * right_iso[m]: packed isometry (table m, site L-1-m) -> table m+1.
 * Tables are host int64; isometry data are host (on_device = 0) or device pointers;
 * they are copied. */
int dmrg_set_mps(dmrg_ctx *ctx, int bond,
                 const int64_t *const *left_tables, const int64_t *left_rows,
                 const double *const *left_iso,
                 const int64_t *const *right_tables, const int64_t *right_rows,
                 const double *const *right_iso, int on_device);

/* SURVEY.md 8(a) a9 looped + a2 + a3: renormalize from both edges to the bond given to
 * dmrg_set_mps, then build the H_eff plan (tables, contracted operators) for it.  `precision` / `slices` select the
 * arithmetic of the rotations (see dmrg_renormalize) and the mode the H_eff plan is prepared for. */
int dmrg_build_env(dmrg_ctx *ctx, int precision, int slices);

/* Split and truncate (PAPER.md:49 truncation error, PAPER.md:51 fixed number of
 * kept states): from the two-site vector psi of the current bond (packed, device pointer if on_device != 0, else
 * host) form the reduced density matrix of the grown block per symmetry sector, eigen-decompose it (host, cyclic
 * Jacobi, FP64), keep the max_states largest weights over all sectors (ties: sector label ascending, then
 * eigen-index) and build the isometry.  direction = DMRG_LEFT_TO_RIGHT grows the left block by site p,
 * DMRG_RIGHT_TO_LEFT the right block by site p+1.  *discarded receives the sum of the dropped weights (for a
 * normalised psi: the truncation error).  The results stay in the context until the next split:
 * dmrg_split_result lends the new bond table (rows of (N, S, dim, offset)) and the isometry in the packed layout
 * that dmrg_renormalize and dmrg_set_mps take (host pointers, borrowed).  Synchronises when psi is on the device.
 * Support step, not timed; SU(2) weights are the eigenvalues in the reduced basis (one per multiplet). */
int dmrg_split_truncate(dmrg_ctx *ctx, const double *psi, int on_device, int direction, int64_t max_states,
                        double *discarded);
int dmrg_split_result(dmrg_ctx *ctx, const int64_t **table, int64_t *table_rows, const double **isometry,
                      int64_t *isometry_len);

/* Two-site DMRG sweeps on the device: from the right-canonical state
 * given to dmrg_set_mps at bond 0 (left tables = the vacuum row only), n_sweeps times rightwards over the bonds
 * 0 .. L-2 and back.  Every bond: H_eff plan, Davidson (`davidson_iters` <= 32 per restart, at most
 * `max_restarts`, until the residual norm is below `tol`) from a random start drawn from `seed`, split and
 * truncate to `max_states` (dmrg_split_truncate), one renormalization.  The operator blocks of both sides stay
 * resident on the device (one stack per side).  energies[] receives the Ritz value + e_core of every bond solve
 * (*n_energies: capacity in, count out, 2 (L-1) per sweep run -- fewer sweeps than n_sweeps when the option sweep_eps
 * stops them); *max_discarded the largest truncation error.  The
 * context is left with the final state and no environments: call dmrg_set_mps / dmrg_build_env to continue. */
int dmrg_sweep(dmrg_ctx *ctx, int n_sweeps, int64_t max_states, int davidson_iters, int max_restarts, double tol,
               int precision, int slices, uint64_t seed, double *energies, int64_t *n_energies, double *max_discarded);

/* Re-plan the current bond for a precision mode (DMRG_PREC_FP64, or DMRG_PREC_FP64_EMU with `slices` = kappa in
 * [2, 7], 0 = 6): which stage-1 jobs and stage-2 segments run on the INT8 tensor cores is a property of the
 * plan.  dmrg_heff_apply / dmrg_davidson_step do this themselves when the mode of a call
 * differs from the plan's; the explicit call exists for planning contexts (tables of an emulated plan without a
 * GPU) and to take the re-planning and operator slicing out of a timed region.  Needs dmrg_build_env or
 * dmrg_plan_bond first. */
int dmrg_replan(dmrg_ctx *ctx, int precision, int slices);

/* Planning only (works without a GPU): build the symmetry tables and launch plans of the
 * bond given to dmrg_set_mps without touching operator data. */
int dmrg_plan_bond(dmrg_ctx *ctx);

int dmrg_psi_length(dmrg_ctx *ctx, int64_t *n);

/* SURVEY.md 8(a) a5 + a6: psi_out = H_eff psi_in (e_core not included); device pointers,
 * packed psi layout, psi_in != psi_out.  Enqueued on the stream, does not synchronise.
 * slices = kappa for DMRG_PREC_FP64_EMU (0 = default 6), ignored otherwise. */
int dmrg_heff_apply(dmrg_ctx *ctx, const double *psi_in_dev, double *psi_out_dev,
                    int precision, int slices);
/* Same through HOST buffers: copies psi_in to the device, applies, copies psi_out back and
 * synchronises (the end-to-end leg of bench.py). */
int dmrg_heff_apply_host(dmrg_ctx *ctx, const double *psi_in_host, double *psi_out_host,
                         int precision, int slices);

/* exact diagonal of H_eff (device pointer, packed psi layout). */
int dmrg_heff_diag(dmrg_ctx *ctx, double *diag_out_dev);

/* Davidson without restart, at most n_iter applications of
 * H_eff starting from psi_inout (device).  tol <= 0 disables the early exit.  On return
 * psi_inout holds the normalised Ritz vector; theta_host[it], resid_host[it] (host arrays of
 * length n_iter) hold the Ritz value and residual norm of iteration it; *n_done the number
 * of applications performed.  Synchronises. */
int dmrg_davidson_step(dmrg_ctx *ctx, double *psi_inout_dev, int n_iter, double tol,
                       int precision, int slices, double *theta_host, double *resid_host,
                       int *n_done);

/* absorb one site into a block.  LEFT_TO_RIGHT: the left block absorbs
 * site `bond`; RIGHT_TO_LEFT: the right block absorbs site bond+1.  new_table: the grown
 * block's bond table (host int64 rows); isometry: packed (old table, site) -> new table
 * (host or device).  The grown block's operator set replaces the previous one; the H_eff
 * plan of the old bond is dropped. */
int dmrg_renormalize(dmrg_ctx *ctx, int direction, const int64_t *new_table, int64_t new_rows,
                     const double *isometry, int on_device, int precision, int slices);
/* (precision: DMRG_PREC_FP64 runs the two rotation products O' = sum f X^T O X on the FP64 tensor pipe;
 * DMRG_PREC_FP64_EMU runs them Ozaki-emulated on the INT8 tensor cores with `slices` = kappa in [2, 7], 0 = 6
 * (all GEMMs emulated), error <= 1e-10 per element relative to the block's largest; DMRG_PREC_TF32X3 runs
 * them as 3xTF32, error <= 1e-5.  The integral-weighted sums of operators (a3) are native FP64 in every mode.) */

/* Borrowed pointer to an int64 table, valid until the next call that changes the plan. */
int dmrg_table(dmrg_ctx *ctx, int which, const int64_t **data, int64_t *count);

/* Parity hook: copy one stored operator of a block to the host as a dense (dim x dim) row-major
 * matrix in the block's bond-table ordering (side 0 = left, 1 = right).  Synchronises. */
int dmrg_op_export(dmrg_ctx *ctx, int side, int kind, int i, int k, double *dense_out_host,
                   int64_t dim);

/* Parity hook for the sampled full-size checks ("taking the environment operator blocks ... as
 * input data downloaded from the device"): copy the stored blocks <i_bra| O |i_ket> of EVERY operator of one class
 * (`kind`, with kind | (2k << 8) for the SU(2) A and B classes; U1U1: the class is (kind, dN, d2Sz) of the operator
 * (i0, k0), any member of it) to the host as out_host[n_members][rows][cols], row-major, and the member labels as
 * members_host[n_members][2] = (i, k) (-1 for unused indices).  Both buffers are caller-owned; `capacity` = doubles
 * available in out_host, `member_capacity` = rows available in members_host.  *n_members, *rows, *cols receive the
 * shape; *n_members = 0 when the class stores no block for this sector pair.  With out_host = NULL only the shape is
 * returned.  Synchronises. */
int dmrg_op_export_class(dmrg_ctx *ctx, int side, int kind, int i0, int k0, int i_bra, int i_ket,
                         double *out_host, int64_t capacity, int64_t *members_host, int64_t member_capacity,
                         int64_t *n_members, int64_t *rows, int64_t *cols);

/* Milliseconds of device time of the last dmrg_heff_apply per stage (stage 1, stage 2) measured with
 * CUDA events when timing is enabled with dmrg_set_timing(ctx, 1).  Synchronises. */
int dmrg_set_timing(dmrg_ctx *ctx, int enable);
int dmrg_last_stage_ms(dmrg_ctx *ctx, double *ms_stage1, double *ms_stage2);
/* Emulated mode only: the part of stage 2 spent slicing T (row a4) and in the tcgen05 INT8 kernel (row a6);
 * both are zero after a native FP64 apply. */
int dmrg_last_emu_ms(dmrg_ctx *ctx, double *ms_slice, double *ms_int8);
/* ... and the part of stage 1 spent in its tensor-core kernel (k_emu_s1 / k_emu_seg / k_tf32_seg; rows a4 + a5): the
 * rest of the stage-1 time is the native FP64 kernel on the jobs below the size thresholds. */
int dmrg_last_emu_stage1_ms(dmrg_ctx *ctx, double *ms_tensor);

/* Micro-benchmarks that measure this GPU's sustained tensor-pipe peaks with the library's own
 * full-tile kernels (SURVEY.md 8(d) "Peaks to measure"): which = DMRG_PREC_*, or 3 = the FP64 vector (non-tensor) FMA
 * rate, the unit on which the emulated epilogue recombines its INT32 sums.
 * Returns operations per second (flop/s for FP64 and 3, int8 op/s for EMU).  Synchronises. */
int dmrg_measure_peak(dmrg_ctx *ctx, int which, double *ops_per_s);

/* Ozaki-emulated FP64 GEMM on the INT8 tensor cores:
 * C[M][N] = A[M][K] B[K][N], row-major device arrays, `slices` = kappa in [2, 7] (0 = 6), triangular
 * product set s + t <= kappa + 1.  This is the contraction engine of DMRG_PREC_FP64_EMU; it is exported
 * so that its numerics (bit-exact slices, INT32 partial sums, <= 1e-10 against FP64) and its tensor-pipe
 * rate can be tested on their own.  ms_slice / ms_gemm (may be NULL) receive device times.  Synchronises. */
int dmrg_emu_gemm(dmrg_ctx *ctx, int M, int N, int K, const double *A_dev, const double *B_dev, double *C_dev,
                  int slices, double *ms_slice, double *ms_gemm);
/* The same product with the slice products cut to s + t <= keep + 1 (1 <= keep <= slices; the operands stay sliced
 * into `slices` digits): the arithmetic of one task class in DMRG_PREC_FP64_EMU_PERF, bit for bit what
 * oracle/ozaki.py emulated_gemm(keep=) models.  Synchronises. */
int dmrg_emu_gemm_kept(dmrg_ctx *ctx, int M, int N, int K, const double *A_dev, const double *B_dev, double *C_dev,
                       int slices, int keep);
/* C[M][N] = sum_g alpha[g] A_g[M][K] B_g[K][N] (A_dev = n stacked row-major matrices, likewise B_dev; alpha on the host;
 * K <= 16384) in DMRG_PREC_FP64_EMU_PERF arithmetic: one task class per g, slice counts chosen on the device by the
 * kernel H_eff.psi uses (k_emu_choose) and returned in keep_out_host[n]; the model is oracle/ozaki.py emulated_sum.
 * Synchronises. */
int dmrg_emu_sum_perf(dmrg_ctx *ctx, int M, int N, int K, int n, const double *A_dev, const double *B_dev,
                      const double *alpha_host, double *C_dev, int slices, int kmin, int32_t *keep_out_host);
/* The performant-mode rule on its own (host arrays, no GPU needed): class i of one job has the magnitude exponents
 * E_all[i] (every line) and E_nz[i] (lines with a non-zero exponent; DMRG_EMU_NO_REF if there is none); keep_out[i]
 * = slices - min(slices - kmin, max(0, max_j E_nz[j] - E_all[i]) / 8), or `slices` when no class has an E_nz. */
#define DMRG_EMU_NO_REF (-(1 << 28))
int dmrg_emu_keep_rule(dmrg_ctx *ctx, const int32_t *E_all, const int32_t *E_nz, int n, int slices, int kmin,
                       int32_t *keep_out);
/* Kernels this context has launched so far (cumulative; the micro-benchmarks of dmrg_measure_peak are not counted): the
 * difference across a timed region is bench.py's `gpu_launches`.  Does not synchronise. */
int dmrg_launch_count(dmrg_ctx *ctx, uint64_t *n);
/* Slice products (x k steps x output tiles) the last DMRG_PREC_FP64_EMU_PERF apply formed in stage 2, and what the
 * eager mode forms on the same segments.  Synchronises. */
int dmrg_last_emu_products(dmrg_ctx *ctx, uint64_t *kept, uint64_t *eager);
/* Row a4 of DMRG_PREC_TF32X3 on its own (reading s15): hi[i] = tf32(x[i]), lo[i] = tf32(x[i] - hi[i]) as FP32
 * bit patterns (device arrays of n elements) -- the split the slicing kernel and the stage-1 epilogue apply; the model is
 * oracle/ozaki.py tf32_split, bit for bit.  Synchronises. */
int dmrg_tf32_split(dmrg_ctx *ctx, const double *src_dev, int64_t n, uint32_t *hi_dev, uint32_t *lo_dev);
/* Row a4 on its own: slice `lines` lines of length K (element (line, k) at src_dev[line * line_stride +
 * k * k_stride]) into out_dev[slices][lines][K] (int8, top digit first) and expo_dev[lines] (int32). */
int dmrg_emu_slice(dmrg_ctx *ctx, const double *src_dev, int lines, int K, int64_t line_stride, int64_t k_stride,
                   int slices, signed char *out_dev, int *expo_dev);

/* The HBM-bound kernels of the path, each timed alone (CUDA events, mean of 5 launches after a warm-up) on the current
 * plan, with the ALGORITHMIC bytes of one launch (north_star "achieved HBM GB/s"): ms_out[i] and
 * bytes_out[i] for i = DMRG_HBM_* below; entries that do not exist in the current plan stay 0.  n_basis (<= 32) is
 * the number of basis vectors of the Davidson kernels (a8).  The slicing kernels (a4) are reported when the plan is in
 * a tensor-core mode (dmrg_replan first): bytes = 8 B read + kappa B (or 8 B for 3xTF32) written per element.
 * Allocates a scratch of (2 n_basis + 4) vectors; psi_dev is read only.  Synchronises. */
enum { DMRG_HBM_DIAG = 0,       /* k_heff_diag (a7): writes diag(H_eff), reads the operator diagonals            */
       DMRG_HBM_DOTS = 1,       /* n_basis dot products V^T w (a8)                                               */
       DMRG_HBM_RITZ = 2,       /* x = V y, r = W y - theta x (a8)                                               */
       DMRG_HBM_PRECOND = 3,    /* t = r / (theta - diag) (a8)                                                   */
       DMRG_HBM_PROJECT = 4,    /* t -= V c (a8, Gram-Schmidt)                                                   */
       DMRG_HBM_SLICE_PSI = 5,  /* slice-and-pack of psi (a4, every apply)                                       */
       DMRG_HBM_SLICE_OPS_L = 6,/* slice-and-pack of the left operators (a4, once per bond)                      */
       DMRG_HBM_SLICE_OPS_R = 7,/* ... of the right operators                                                    */
       DMRG_HBM_SLICE_T = 8,    /* slice-and-pack of the part of T that the stage-1 epilogue does not emit (a4)  */
       DMRG_HBM_N = 9 };
int dmrg_measure_hbm_kernels(dmrg_ctx *ctx, const double *psi_dev, int n_basis, double *ms_out, double *bytes_out,
                             int capacity, int *n_out);

/* Row a8 building block on its own, through the context: out_dev[v] = <V_v, w>, v < nvec <= 32, V_v = V_dev + v * ld,
 * vectors of length n (the Gram-matrix column and Gram-Schmidt projections of the Davidson step, SURVEY.md 8(a) a8,
 * 8(c) c6).  Device pointers; enqueued on the context's stream; partial sums go through the context's own buffer. */
int dmrg_dots(dmrg_ctx *ctx, const double *V_dev, int64_t ld, int nvec, const double *w_dev, int64_t n,
              double *out_dev);

/* The same dot products for callers that may not allocate device memory (code under CUDA graph capture, serving
 * loops, harnesses that forbid cudaMalloc): needs no context and calls no cudaMalloc / cudaFree or allocating
 * library routine.  The per-block partial sums live in a static device array inside the library (32 x 296 doubles =
 * 74 KB, held by every GPU that loads the library until the process exits), so nvec must be in [1, 32] (else
 * DMRG_EINVAL with a message); n is unlimited.  Runs on the CURRENT device, on `cuda_stream` (a cudaStream_t as
 * void*, NULL = default stream), does not synchronise, and gives bit-identical results to dmrg_dots (same kernels,
 * same summation order).  All calls on one GPU share the array: calls that overlap on the GPU (different streams)
 * race on it -- serialise them.  Nothing in it has to be cleared between calls: every entry read is written first.
 * Returns DMRG_OK or a negative code; dmrg_noalloc_last_error() gives the message of the calling thread's last
 * failure (borrowed). */
int dmrg_dots_noalloc(void *cuda_stream, const double *V_dev, int64_t ld, int nvec, const double *w_dev, int64_t n,
                      double *out_dev);
const char *dmrg_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
